// gabsplat_render_host: the four calls of the ABI chained for a caller whose buffers live in HOST memory
// (the end-to-end leg of bench.py).  Only copies and calls of the public entry points; no kernels here.
#include <cstdio>

#include "common.cuh"

namespace {

using namespace gabsplat;

struct Arena {
  char* base;
  uint64_t off;
  template <typename T>
  T* take(uint64_t n) {
    T* p = reinterpret_cast<T*>(base + off);
    off = (off + n * sizeof(T) + 255) / 256 * 256;
    return p;
  }
};

struct Layout {
  gabsplat_scene scene;
  gabsplat_projected proj;
  gabsplat_binning bin;
  gabsplat_fwd_out fwd;
  gabsplat_grads grads;
  float* dL;
  void* grad_ws;
  uint64_t grad_ws_bytes;
  uint64_t bytes;
};

Layout carve(void* base, int N, int K, int width, int height, uint64_t capacity) {
  Arena a{(char*)base, 0};
  Layout l;
  const uint64_t n = (uint64_t)N, k = (uint64_t)K, hw = (uint64_t)width * height;
  const uint64_t tiles = (uint64_t)((width + kTile - 1) / kTile) * ((height + kTile - 1) / kTile);
  l.scene.N = N; l.scene.K = K; l.scene.sh_degree = 3;
  l.scene.means = a.take<float>(n * 3);
  l.scene.scales = a.take<float>(n * 3);
  l.scene.rotations = a.take<float>(n * 4);
  l.scene.opacities = a.take<float>(n);
  l.scene.sh = a.take<float>(n * 48);
  l.scene.freqs = a.take<float>(n * k * 3);
  l.scene.weights = a.take<float>(n * k);
  l.proj.mean2d = a.take<float>(n * 2);
  l.proj.depth = a.take<float>(n);
  l.proj.radius = a.take<int32_t>(n);
  l.proj.conic_opacity = a.take<float>(n * 4);
  l.proj.rgb = a.take<float>(n * 3);
  l.proj.rgb_clamped = a.take<uint8_t>(n * 4);
  l.proj.freq2d = a.take<float>(n * k * 2);
  l.proj.tiles_touched = a.take<uint32_t>(n);
  l.proj.rect = a.take<int32_t>(n * 4);
  l.proj.packed = a.take<float>(n * packed_floats(K));
  l.proj.chunk_visible = a.take<uint32_t>(gabsplat_chunk_visible_count(N));
  l.bin.offsets = a.take<uint32_t>(n);
  l.bin.keys = a.take<uint64_t>(capacity);
  l.bin.ids = a.take<uint32_t>(capacity);
  l.bin.tile_ranges = a.take<uint32_t>(tiles * 2);
  l.bin.tile_order = a.take<uint32_t>(tiles);
  l.bin.capacity = capacity;
  l.bin.num_instances = a.take<uint32_t>(4);
  l.bin.workspace_bytes = sort_workspace_bytes(N, capacity, (int)tiles);
  l.bin.workspace = a.take<char>(l.bin.workspace_bytes);
  l.bin.tile_work_hint = nullptr;
  l.fwd.image = a.take<float>(3 * hw);
  l.fwd.final_T = a.take<float>(hw);
  l.fwd.n_contrib = a.take<uint32_t>(hw);
  l.fwd.blend_state_bytes = blend_state_bytes(tiles, capacity);
  l.fwd.blend_state = a.take<char>(l.fwd.blend_state_bytes);
  l.fwd.tile_work = nullptr;
  l.dL = a.take<float>(3 * hw);
  l.grads.d_means = a.take<float>(n * 3);
  l.grads.d_scales = a.take<float>(n * 3);
  l.grads.d_rotations = a.take<float>(n * 4);
  l.grads.d_opacities = a.take<float>(n);
  l.grads.d_sh = a.take<float>(n * 48);
  l.grads.d_freqs = a.take<float>(n * k * 3);
  l.grads.d_weights = a.take<float>(n * k);
  l.grads.d_mean2d = nullptr;
  l.grads.d_mean2d_abs = nullptr;
  l.grad_ws_bytes = gabsplat_grad_workspace_bytes(N, K);
  l.grad_ws = a.take<char>(l.grad_ws_bytes);
  l.bytes = a.off;
  return l;
}

}  // namespace

extern "C" {

uint64_t gabsplat_host_arena_bytes(int32_t N, int32_t K, int32_t width, int32_t height, uint64_t capacity) {
  if (N < 0 || K < 0 || K > kMaxK || width <= 0 || height <= 0) return 0;
  return carve(nullptr, N, K, width, height, capacity).bytes;
}

int32_t gabsplat_render_host(gabsplat_ctx* ctx, const gabsplat_scene* sh, const gabsplat_camera* cam,
                             uint64_t capacity, float* image_host, const float* dL_dimage_host,
                             gabsplat_grads* gh, void* device_arena, uint64_t arena_bytes, void* stream) {
  if (!ctx || !sh || !cam || !image_host || !device_arena) return GABSPLAT_INVALID_ARG;
  // everything the calls below would refuse is refused here, before a single copy has been queued
  if (!scene_ok(sh) || !camera_ok(cam)) {
    std::snprintf(ctx->error, sizeof(ctx->error), "render_host: bad %s", scene_ok(sh) ? "camera" : "scene");
    return GABSPLAT_INVALID_ARG;
  }
  if (dL_dimage_host && !gh) return GABSPLAT_INVALID_ARG;
  if (dL_dimage_host && sh->N > 0 &&
      (!gh->d_means || !gh->d_scales || !gh->d_rotations || !gh->d_opacities || !gh->d_sh || (sh->K > 0 && (!gh->d_freqs || !gh->d_weights))))
    return GABSPLAT_INVALID_ARG;
  if (((uintptr_t)device_arena & 255) != 0) return GABSPLAT_INVALID_ARG;
  Layout l = carve(device_arena, sh->N, sh->K, cam->width, cam->height, capacity);
  if (arena_bytes < l.bytes) return GABSPLAT_CAPACITY;
  l.scene.sh_degree = sh->sh_degree;
  cudaStream_t st = (cudaStream_t)stream, cin = ctx->copy_in, cout = ctx->copy_out;
  const uint64_t n = (uint64_t)sh->N, k = (uint64_t)sh->K, hw = (uint64_t)cam->width * cam->height, f = sizeof(float);
  // Uploads run on a copy stream in the order the kernels need them, downloads on another; the kernels wait for exactly
  // the arrays they read:
  //   means, scales, rotations (40 B per primitive)  -> the indexing track and the whole binning start
  //   opacities, frequencies, weights, SH colours    -> the value track (side stream, beside the binning), the blends
  //   dL/dimage                                      -> the backward
  //   image                                          <- leaves while the backward runs
  // A failure after this point leaves with copies from / to the caller's host buffers possibly still in flight on the two
  // internal streams, which the caller cannot wait for: every error return drains them (and the caller's stream) first.
  auto bail = [&](int32_t rc) {
    cudaStreamSynchronize(cin);
    cudaStreamSynchronize(cout);
    cudaStreamSynchronize(st);
    return rc;
  };
#define GS_CK(call) if ((call) != cudaSuccess) return bail(GABSPLAT_CUDA)
#define GS_H2D(dst, src, count) if (count) GS_CK(cudaMemcpyAsync((void*)(dst), (src), (count) * f, cudaMemcpyHostToDevice, cin))
#define GS_D2H(dst, src, count, s) if (count) GS_CK(cudaMemcpyAsync((dst), (const void*)(src), (count) * f, cudaMemcpyDeviceToHost, s))
  GS_CK(cudaEventRecord(ctx->ev_copy[0], st));          // whatever the caller queued before this call
  GS_CK(cudaStreamWaitEvent(cin, ctx->ev_copy[0], 0));
  GS_CK(cudaStreamWaitEvent(cout, ctx->ev_copy[0], 0));
  GS_H2D(l.scene.means, sh->means, n * 3);
  GS_H2D(l.scene.scales, sh->scales, n * 3);
  GS_H2D(l.scene.rotations, sh->rotations, n * 4);
  GS_CK(cudaEventRecord(ctx->ev_copy[1], cin));
  GS_H2D(l.scene.opacities, sh->opacities, n);
  GS_H2D(l.scene.freqs, sh->freqs, n * k * 3);
  GS_H2D(l.scene.weights, sh->weights, n * k);
  GS_H2D(l.scene.sh, sh->sh, n * 48);
  GS_CK(cudaEventRecord(ctx->ev_copy[2], cin));
  if (dL_dimage_host) {
    GS_H2D(l.dL, dL_dimage_host, 3 * hw);
    GS_CK(cudaEventRecord(ctx->ev_copy[3], cin));
  }
  l.scene.variant = sh->variant;
  GS_CK(cudaStreamWaitEvent(st, ctx->ev_copy[1], 0));
  int32_t rc = gabsplat_preprocess_bin_sort_ordered(ctx, &l.scene, cam, &l.proj, &l.bin, nullptr, stream, ctx->ev_copy[2]);
  if (rc != GABSPLAT_OK) return bail(rc);
  if (!dL_dimage_host) l.fwd.blend_state = nullptr;  // inference: nothing to replay
  rc = gabsplat_render_forward(ctx, &l.scene, cam, &l.proj, &l.bin, &l.fwd, stream);
  if (rc != GABSPLAT_OK) return bail(rc);
  GS_CK(cudaEventRecord(ctx->ev_copy[4], st));
  GS_CK(cudaStreamWaitEvent(cout, ctx->ev_copy[4], 0));
  GS_D2H(image_host, l.fwd.image, 3 * hw, cout);
  uint32_t* count_slot = reinterpret_cast<uint32_t*>(ctx->pinned_count);
  GS_CK(cudaMemcpyAsync(count_slot, l.bin.num_instances, sizeof(uint32_t), cudaMemcpyDeviceToHost, cout));
  if (dL_dimage_host) {
    GS_CK(cudaStreamWaitEvent(st, ctx->ev_copy[3], 0));
    rc = gabsplat_render_backward(ctx, &l.scene, cam, &l.proj, &l.bin, &l.fwd, l.dL, &l.grads, l.grad_ws,
                                  l.grad_ws_bytes, stream);
    if (rc != GABSPLAT_OK) return bail(rc);
    GS_D2H(gh->d_means, l.grads.d_means, n * 3, st);
    GS_D2H(gh->d_scales, l.grads.d_scales, n * 3, st);
    GS_D2H(gh->d_rotations, l.grads.d_rotations, n * 4, st);
    GS_D2H(gh->d_opacities, l.grads.d_opacities, n, st);
    GS_D2H(gh->d_sh, l.grads.d_sh, n * 48, st);
    GS_D2H(gh->d_freqs, l.grads.d_freqs, n * k * 3, st);
    GS_D2H(gh->d_weights, l.grads.d_weights, n * k, st);
  }
#undef GS_H2D
#undef GS_D2H
  // the caller's stream ends after everything this call queued anywhere
  GS_CK(cudaEventRecord(ctx->ev_copy[0], cout));
  GS_CK(cudaStreamWaitEvent(st, ctx->ev_copy[0], 0));
  GS_CK(cudaEventRecord(ctx->ev_copy[1], cin));
  GS_CK(cudaStreamWaitEvent(st, ctx->ev_copy[1], 0));
  GS_CK(cudaStreamSynchronize(st));
#undef GS_CK
  // an instance list larger than `capacity` renders the background only (every stage checks the count on the device)
  if ((uint64_t)*count_slot > capacity) return GABSPLAT_CAPACITY;
  return GABSPLAT_OK;
}

}  // extern "C"
