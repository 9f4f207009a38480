// The C ABI of libgabsplat (include/gabsplat.h): argument checking, status codes, and the order of
// kernel launches.  No arithmetic of the method lives here.
#include <cstdio>
#include <cstring>
#include <new>

#include "common.cuh"

namespace gabsplat {
std::atomic<unsigned long long> g_kernel_launches{0};

// argument checks shared with host_api.cu (which must refuse a bad scene before it queues the first copy)
bool camera_ok(const gabsplat_camera* c) {
  // z_near > 0 (also rejects NaN): the depth key orders bits(t_z) as unsigned integers, valid for positive floats only
  return c && c->width > 0 && c->height > 0 && c->fx > 0.f && c->fy > 0.f && c->z_near > 0.f &&
         (int64_t)((c->width + kTile - 1) / kTile) * ((c->height + kTile - 1) / kTile) < (1 << 30);
}

bool scene_ok(const gabsplat_scene* s) {
  if (!s || s->N < 0 || s->K < 0 || s->K > kMaxK || s->sh_degree < 0 || s->sh_degree > 3 || s->variant < 0 || s->variant > 3) return false;
  if (s->N == 0) return true;
  if (!s->means || !s->scales || !s->rotations || !s->opacities || !s->sh) return false;
  if (s->K > 0 && (!s->freqs || !s->weights)) return false;
  return true;
}
}  // namespace gabsplat

namespace {

using namespace gabsplat;

int32_t fail(gabsplat_ctx* ctx, int32_t code, const char* msg) {
  if (ctx) {
    std::strncpy(ctx->error, msg, sizeof(ctx->error) - 1);
    ctx->error[sizeof(ctx->error) - 1] = 0;
  }
  return code;
}

int32_t cuda_fail(gabsplat_ctx* ctx, cudaError_t e, const char* where) {
  if (ctx) std::snprintf(ctx->error, sizeof(ctx->error), "%s: %s", where, cudaGetErrorString(e));
  return GABSPLAT_CUDA;
}

bool projected_ok(const gabsplat_projected* p, int N, int K) {
  if (!p) return false;
  if (N == 0) return true;
  return p->mean2d && p->depth && p->radius && p->conic_opacity && p->rgb && p->rgb_clamped &&
         (K == 0 || p->freq2d) && p->tiles_touched && p->rect && p->packed && p->chunk_visible;
}

bool binning_ok(const gabsplat_binning* b, int N) {
  if (!b || !b->tile_ranges || !b->tile_order || !b->num_instances) return false;
  if (N > 0 && !b->offsets) return false;
  if (b->capacity > 0 && !b->ids) return false;
  if (b->capacity >= (1ull << 32)) return false;
  return true;
}

}  // namespace

extern "C" {

int32_t gabsplat_create(gabsplat_ctx** out, int32_t device) {
  if (!out) return GABSPLAT_INVALID_ARG;
  *out = nullptr;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
    cudaGetLastError();
    return GABSPLAT_UNSUPPORTED;
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return GABSPLAT_CUDA;
  if (prop.major != 10) return GABSPLAT_UNSUPPORTED;  // the kernels are built for sm_100a only
  if (cudaSetDevice(device) != cudaSuccess) return GABSPLAT_CUDA;
  gabsplat_ctx* ctx = new (std::nothrow) gabsplat_ctx;
  if (!ctx) return GABSPLAT_CUDA;
  ctx->device = device;
  ctx->error[0] = 0;
  ctx->pinned_count = nullptr;
  if (cudaMallocHost(&ctx->pinned_count, sizeof(uint64_t)) != cudaSuccess) {
    delete ctx;
    return GABSPLAT_CUDA;
  }
  ctx->side = nullptr; ctx->ev_fork = ctx->ev_join = nullptr; ctx->scratch = nullptr;
  ctx->copy_in = ctx->copy_out = nullptr;
  for (cudaEvent_t& e : ctx->ev_copy) e = nullptr;
  ctx->place_bands = 0;
  bool ok = cudaStreamCreateWithFlags(&ctx->copy_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&ctx->copy_out, cudaStreamNonBlocking) == cudaSuccess;
  for (cudaEvent_t& e : ctx->ev_copy) ok = ok && cudaEventCreateWithFlags(&e, cudaEventDisableTiming) == cudaSuccess;
  if (!ok || cudaMalloc(&ctx->scratch, 256) != cudaSuccess ||
      cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) != cudaSuccess) {
    gabsplat_destroy(ctx);
    return GABSPLAT_CUDA;
  }
  cudaDeviceSynchronize();
  *out = ctx;
  return GABSPLAT_OK;
}

void gabsplat_destroy(gabsplat_ctx* ctx) {
  if (!ctx) return;
  if (ctx->pinned_count) cudaFreeHost(ctx->pinned_count);
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
  if (ctx->side) cudaStreamDestroy(ctx->side);
  if (ctx->copy_in) cudaStreamDestroy(ctx->copy_in);
  if (ctx->copy_out) cudaStreamDestroy(ctx->copy_out);
  for (cudaEvent_t e : ctx->ev_copy) if (e) cudaEventDestroy(e);
  if (ctx->scratch) cudaFree(ctx->scratch);
  ctx->timer.destroy();
  delete ctx;
}

const char* gabsplat_last_error(const gabsplat_ctx* ctx) { return ctx ? ctx->error : "null context"; }

int32_t gabsplat_packed_floats(int32_t K) { return (K < 0 || K > kMaxK) ? 0 : packed_floats(K); }

uint64_t gabsplat_sort_workspace_bytes(int32_t N, uint64_t capacity, int32_t width, int32_t height) {
  if (width <= 0 || height <= 0) return 0;
  return sort_workspace_bytes(N < 0 ? 0 : N, capacity, ((width + kTile - 1) / kTile) * ((height + kTile - 1) / kTile));
}

uint64_t gabsplat_blend_state_bytes(int32_t width, int32_t height, uint64_t capacity) {
  if (width <= 0 || height <= 0) return 0;
  return blend_state_bytes((uint64_t)((width + kTile - 1) / kTile) * ((height + kTile - 1) / kTile), capacity);
}

uint64_t gabsplat_grad_workspace_bytes(int32_t N, int32_t K) {
  if (N < 0 || K < 0 || K > kMaxK) return 0;
  return (uint64_t)N * grad2d_floats(K) * sizeof(float) + 256;
}

int32_t gabsplat_preprocess(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                            gabsplat_projected* out, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (!scene_ok(scene)) return fail(ctx, GABSPLAT_INVALID_ARG, "preprocess: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "preprocess: bad camera");
  if (!projected_ok(out, scene->N, scene->K)) return fail(ctx, GABSPLAT_INVALID_ARG, "preprocess: null output");
  ctx->timer.begin(GABSPLAT_STAGE_PREPROCESS, (cudaStream_t)stream);
  const cudaError_t e = launch_preprocess(*scene, make_camera(*cam), *out, (cudaStream_t)stream, (cudaStream_t)stream, nullptr);
  ctx->timer.end((cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "preprocess");
}

int32_t gabsplat_preprocess_bin_sort(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                     gabsplat_projected* proj, gabsplat_binning* bin, uint64_t* num_instances_host,
                                     void* stream) {
  return gabsplat_preprocess_bin_sort_ordered(ctx, scene, cam, proj, bin, num_instances_host, stream, nullptr);
}

}  // extern "C"

int32_t gabsplat_preprocess_bin_sort_ordered(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                             gabsplat_projected* proj, gabsplat_binning* bin, uint64_t* num_instances_host,
                                             void* stream, cudaEvent_t value_inputs_ready) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  // with the stage timer on, or nothing to overlap, this is exactly the two calls
  if (ctx->timer.on || !scene || scene->N <= 0) {
    if (value_inputs_ready && cudaStreamWaitEvent((cudaStream_t)stream, value_inputs_ready, 0) != cudaSuccess) return GABSPLAT_CUDA;
    const int32_t rc = gabsplat_preprocess(ctx, scene, cam, proj, stream);
    return rc != GABSPLAT_OK ? rc : gabsplat_bin_sort(ctx, scene->N, proj, cam, bin, num_instances_host, stream);
  }
  if (!scene_ok(scene)) return fail(ctx, GABSPLAT_INVALID_ARG, "preprocess_bin_sort: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "preprocess_bin_sort: bad camera");
  if (!projected_ok(proj, scene->N, scene->K)) return fail(ctx, GABSPLAT_INVALID_ARG, "preprocess_bin_sort: null output");
  cudaStream_t st = (cudaStream_t)stream;
  // the binning needs only the indexing track: the fp64 value track runs on the side stream beside it
  cudaError_t e = value_inputs_ready ? cudaStreamWaitEvent(ctx->side, value_inputs_ready, 0) : cudaSuccess;
  if (e == cudaSuccess) e = launch_preprocess(*scene, make_camera(*cam), *proj, st, ctx->side, ctx->ev_fork);
  if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_join, ctx->side);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "preprocess_bin_sort (projection)");
  const int32_t rc = gabsplat_bin_sort(ctx, scene->N, proj, cam, bin, num_instances_host, stream);
  e = cudaStreamWaitEvent(st, ctx->ev_join, 0);  // join even when the binning reported an error
  if (e != cudaSuccess) return cuda_fail(ctx, e, "preprocess_bin_sort (join)");
  return rc;
}

extern "C" {

int32_t gabsplat_bin_sort(gabsplat_ctx* ctx, int32_t N, const gabsplat_projected* proj, const gabsplat_camera* cam,
                          gabsplat_binning* bin, uint64_t* num_instances_host, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (N < 0 || !camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "bin_sort: bad N or camera");
  if (!proj || (N > 0 && (!proj->tiles_touched || !proj->rect || !proj->depth || !proj->chunk_visible)))
    return fail(ctx, GABSPLAT_INVALID_ARG, "bin_sort: null projected arrays");
  if (!binning_ok(bin, N)) return fail(ctx, GABSPLAT_INVALID_ARG, "bin_sort: bad binning buffers");
  if (bin->capacity > 0 && !bin->keys && !keys_optional(((cam->width + kTile - 1) / kTile) * ((cam->height + kTile - 1) / kTile)))
    return fail(ctx, GABSPLAT_INVALID_ARG, "bin_sort: images of more than 26000 tiles need the key buffer");
  if (!bin->workspace ||
      bin->workspace_bytes < gabsplat_sort_workspace_bytes(N, bin->capacity, cam->width, cam->height))
    return fail(ctx, GABSPLAT_CAPACITY, "bin_sort: workspace too small");
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = launch_bin_sort(N, *proj, make_camera(*cam), *bin, ctx->timer, ctx->place_bands, st);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "bin_sort");
  if (num_instances_host) {
    uint32_t* slot = reinterpret_cast<uint32_t*>(ctx->pinned_count);
    e = cudaMemcpyAsync(slot, bin->num_instances, sizeof(uint32_t), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "bin_sort readback");
    *num_instances_host = *slot;
    if (*num_instances_host > bin->capacity) return fail(ctx, GABSPLAT_CAPACITY, "bin_sort: instance capacity too small");
  }
  return GABSPLAT_OK;
}

int32_t gabsplat_render_forward(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                const gabsplat_projected* proj, const gabsplat_binning* bin, gabsplat_fwd_out* out,
                                void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (!scene || scene->K < 0 || scene->K > kMaxK || scene->N < 0) return fail(ctx, GABSPLAT_INVALID_ARG, "render_forward: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_forward: bad camera");
  if (!proj || (scene->N > 0 && !proj->packed)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_forward: null packed records");
  if (!bin || !bin->tile_ranges || !bin->tile_order || (bin->capacity > 0 && !bin->ids)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_forward: bad binning");
  if (!out || !out->image || !out->final_T || !out->n_contrib) return fail(ctx, GABSPLAT_INVALID_ARG, "render_forward: null output");
  const Camera c = make_camera(*cam);
  const uint64_t tiles = (uint64_t)c.tiles_x * c.tiles_y;
  BlendState save;
  if (out->blend_state) {
    if (out->blend_state_bytes < blend_state_bytes(tiles, bin->capacity))
      return fail(ctx, GABSPLAT_CAPACITY, "render_forward: blend_state too small");
    save = make_blend_state(out->blend_state, tiles, bin->capacity);
  }
  ctx->timer.begin(GABSPLAT_STAGE_BLEND_FORWARD, (cudaStream_t)stream);
  const cudaError_t e = launch_blend_forward(scene->K, c, *proj, *bin, *out, out->blend_state ? &save : nullptr,
                                             (cudaStream_t)stream);
  ctx->timer.end((cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "render_forward");
}

int32_t gabsplat_render_backward(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                 const gabsplat_projected* proj, const gabsplat_binning* bin,
                                 const gabsplat_fwd_out* fwd, const float* dL_dimage, gabsplat_grads* grads,
                                 void* grad_workspace, uint64_t grad_workspace_bytes, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (!scene_ok(scene)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: bad camera");
  if (!projected_ok(proj, scene->N, scene->K)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: null projected arrays");
  if (!bin || !bin->tile_ranges || (bin->capacity > 0 && !bin->ids)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: bad binning");
  if (!fwd || !fwd->final_T || !fwd->n_contrib || !dL_dimage) return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: null forward state");
  if (!fwd->blend_state)
    return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: the forward was run without blend_state (inference mode)");
  if (scene->N > 0 && (!bin->workspace ||
                       bin->workspace_bytes < gabsplat_sort_workspace_bytes(scene->N, bin->capacity, cam->width, cam->height)))
    return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: bin.workspace must still hold what gabsplat_bin_sort left in it");
  if (!grads) return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: null grads");
  if (scene->N > 0 && (!grads->d_means || !grads->d_scales || !grads->d_rotations || !grads->d_opacities || !grads->d_sh ||
                       (scene->K > 0 && (!grads->d_freqs || !grads->d_weights))))
    return fail(ctx, GABSPLAT_INVALID_ARG, "render_backward: null gradient output");
  if (scene->N > 0 && (!grad_workspace || grad_workspace_bytes < gabsplat_grad_workspace_bytes(scene->N, scene->K)))
    return fail(ctx, GABSPLAT_CAPACITY, "render_backward: gradient workspace too small");
  cudaStream_t st = (cudaStream_t)stream;
  const Camera c = make_camera(*cam);
  float* grad2d = reinterpret_cast<float*>(((uintptr_t)grad_workspace + 255) & ~(uintptr_t)255);
  const uint64_t tiles = (uint64_t)c.tiles_x * c.tiles_y;
  if (fwd->blend_state_bytes < blend_state_bytes(tiles, bin->capacity))
    return fail(ctx, GABSPLAT_CAPACITY, "render_backward: blend_state too small");
  const BlendState saved = make_blend_state(fwd->blend_state, tiles, bin->capacity);
  // fork: zero the gradient arrays on the side stream (store-only, HBM bound) while the blend backward
  // (ALU bound) runs on the caller's stream; join before the projection backward writes the visible rows
  cudaError_t e = cudaEventRecord(ctx->ev_fork, st);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0);
  if (e == cudaSuccess) e = launch_grad_zero(*scene, *grads, ctx->side);
  if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_join, ctx->side);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "render_backward (gradient zeroing)");
  ctx->timer.begin(GABSPLAT_STAGE_BLEND_BACKWARD, st);
  e = launch_blend_backward(scene->N, scene->K, grads->d_mean2d_abs != nullptr, c, *proj, *bin, *fwd, saved,
                                        dL_dimage, grad2d, st);
  ctx->timer.end(st);
  // join the side stream on every path: a later call must never race the zeroing of the gradient arrays
  const cudaError_t ej = cudaStreamWaitEvent(st, ctx->ev_join, 0);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "render_backward (blend)");
  if (ej != cudaSuccess) return cuda_fail(ctx, ej, "render_backward (join)");
  ctx->timer.begin(GABSPLAT_STAGE_PREPROCESS_BACKWARD, st);
  e = launch_preprocess_backward(*scene, c, *proj, *bin, grad2d, *grads, st);
  ctx->timer.end(st);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "render_backward (projection)");
}

uint64_t gabsplat_aux_workspace_bytes(int32_t N, int32_t width, int32_t height) {
  if (N < 0 || width <= 0 || height <= 0) return 0;
  return (uint64_t)N * 16 + 256 + (uint64_t)width * height * 8 + 512;
}

int32_t gabsplat_render_aux(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                            const gabsplat_projected* proj, const gabsplat_binning* bin, float* aux_image,
                            void* workspace, uint64_t workspace_bytes, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (!scene_ok(scene)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_aux: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_aux: bad camera");
  if (!projected_ok(proj, scene->N, scene->K)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_aux: null projected arrays");
  if (!bin || !bin->tile_ranges || !bin->tile_order || (bin->capacity > 0 && !bin->ids)) return fail(ctx, GABSPLAT_INVALID_ARG, "render_aux: bad binning");
  if (!aux_image) return fail(ctx, GABSPLAT_INVALID_ARG, "render_aux: null output");
  if (!workspace || workspace_bytes < gabsplat_aux_workspace_bytes(scene->N, cam->width, cam->height))
    return fail(ctx, GABSPLAT_CAPACITY, "render_aux: workspace too small");
  const uint64_t hw = (uint64_t)cam->width * cam->height;
  char* w = reinterpret_cast<char*>(((uintptr_t)workspace + 255) & ~(uintptr_t)255);
  float4* aux = reinterpret_cast<float4*>(w);
  w += ((uint64_t)scene->N * 16 + 255) & ~255ull;
  float* final_T = reinterpret_cast<float*>(w);
  uint32_t* n_contrib = reinterpret_cast<uint32_t*>(w + ((hw * 4 + 255) & ~255ull));
  const cudaError_t e = launch_blend_aux(scene->N, scene->K, scene->weights, make_camera(*cam), *proj, *bin, aux, aux_image,
                                         final_T, n_contrib, (cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "render_aux");
}

uint64_t gabsplat_loss_workspace_bytes(int32_t width, int32_t height) {
  return (width <= 0 || height <= 0) ? 0 : loss_workspace_bytes(width, height);
}

int32_t gabsplat_loss(gabsplat_ctx* ctx, int32_t width, int32_t height, const float* image, const float* target, float lambda,
                      float* loss_out, float* dL_dimage, void* workspace, uint64_t workspace_bytes, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (width <= 0 || height <= 0 || !image || !target || !loss_out || !(lambda >= 0.f && lambda <= 1.f))
    return fail(ctx, GABSPLAT_INVALID_ARG, "loss: bad size, lambda or null pointer");
  if (!workspace || workspace_bytes < loss_workspace_bytes(width, height))
    return fail(ctx, GABSPLAT_CAPACITY, "loss: workspace too small");
  const cudaError_t e = launch_loss(width, height, image, target, lambda, loss_out, dL_dimage, workspace, (cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "loss");
}

uint64_t gabsplat_chunk_visible_count(int32_t N) {
  return N <= 0 ? 1 : 3 * (((uint64_t)N + GABSPLAT_CHUNK - 1) / GABSPLAT_CHUNK) + 1;
}

uint64_t gabsplat_kernel_launches(void) { return g_kernel_launches.load(std::memory_order_relaxed); }

int32_t gabsplat_trace_pixels(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                              const gabsplat_projected* proj, const gabsplat_binning* bin, int32_t n, const int32_t* pixels,
                              const uint32_t* offsets, uint32_t* entries, float* colour_T, uint32_t* info, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (!scene || scene->K < 0 || scene->K > kMaxK || scene->N < 0) return fail(ctx, GABSPLAT_INVALID_ARG, "trace_pixels: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "trace_pixels: bad camera");
  if (!proj || (scene->N > 0 && !proj->packed)) return fail(ctx, GABSPLAT_INVALID_ARG, "trace_pixels: null packed records");
  if (!bin || !bin->tile_ranges || (bin->capacity > 0 && !bin->ids)) return fail(ctx, GABSPLAT_INVALID_ARG, "trace_pixels: bad binning");
  if (n < 0 || (n > 0 && (!pixels || !offsets || !entries || !colour_T || !info)))
    return fail(ctx, GABSPLAT_INVALID_ARG, "trace_pixels: null argument");
  const cudaError_t e = launch_trace_pixels(scene->K, make_camera(*cam), *proj, *bin, n, pixels, offsets, entries, colour_T, info,
                                            (cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "trace_pixels");
}

int32_t gabsplat_probe_sincos(gabsplat_ctx* ctx, int32_t n, const float* phase, float* cos_out, float* sin_out, void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (n < 0 || (n > 0 && (!phase || !cos_out || !sin_out))) return fail(ctx, GABSPLAT_INVALID_ARG, "probe_sincos: null argument");
  const cudaError_t e = launch_probe_sincos(n, phase, cos_out, sin_out, (cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "probe_sincos");
}

int32_t gabsplat_set_place_bands(gabsplat_ctx* ctx, int32_t bands) {
  if (!ctx || bands < 0) return GABSPLAT_INVALID_ARG;
  ctx->place_bands = bands;
  return GABSPLAT_OK;
}

int32_t gabsplat_measure_peaks(gabsplat_ctx* ctx, float* results_host, void* stream) {
  if (!ctx || !results_host) return GABSPLAT_INVALID_ARG;
  const cudaError_t e = measure_peaks(results_host, ctx->scratch, (cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "measure_peaks");
}

int32_t gabsplat_timing_enable(gabsplat_ctx* ctx, int32_t on) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  ctx->timer.on = on != 0;
  ctx->timer.reset();
  return GABSPLAT_OK;
}

int32_t gabsplat_timing_read(gabsplat_ctx* ctx, int32_t* stage_ids_host, float* ms_host, int32_t max_records,
                             int32_t* n_records_host) {
  if (!ctx || !n_records_host || max_records < 0 || (max_records > 0 && (!stage_ids_host || !ms_host)))
    return GABSPLAT_INVALID_ARG;
  StageTimer& tm = ctx->timer;
  *n_records_host = (int32_t)tm.recs.size();
  for (size_t i = 0; i < tm.recs.size() && (int32_t)i < max_records; ++i) {
    cudaError_t e = cudaEventSynchronize(tm.recs[i].b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, tm.recs[i].a, tm.recs[i].b);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "timing_read");
    stage_ids_host[i] = tm.recs[i].stage;
    ms_host[i] = ms;
  }
  tm.reset();
  return GABSPLAT_OK;
}

int32_t gabsplat_count_pairs(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                             const gabsplat_projected* proj, const gabsplat_binning* bin, uint32_t* counters,
                             void* stream) {
  if (!ctx) return GABSPLAT_INVALID_ARG;
  if (!scene || scene->K < 0 || scene->K > kMaxK || scene->N < 0) return fail(ctx, GABSPLAT_INVALID_ARG, "count_pairs: bad scene");
  if (!camera_ok(cam)) return fail(ctx, GABSPLAT_INVALID_ARG, "count_pairs: bad camera");
  if (!proj || (scene->N > 0 && !proj->packed)) return fail(ctx, GABSPLAT_INVALID_ARG, "count_pairs: null packed records");
  if (!bin || !bin->tile_ranges || !bin->tile_order || (bin->capacity > 0 && !bin->ids)) return fail(ctx, GABSPLAT_INVALID_ARG, "count_pairs: bad binning");
  if (!counters) return fail(ctx, GABSPLAT_INVALID_ARG, "count_pairs: null output");
  const cudaError_t e = launch_count_pairs(scene->K, make_camera(*cam), *proj, *bin, counters, (cudaStream_t)stream);
  return e == cudaSuccess ? GABSPLAT_OK : cuda_fail(ctx, e, "count_pairs");
}

}  // extern "C"
