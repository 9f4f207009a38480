// Shared declarations of the CUDA path (libgabsplat.so).  Nothing here is used by oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <vector>

#include "../../include/gabsplat.h"

namespace gabsplat {

// Named constants of the rasterizer the paper adopts from 3DGS (readings C5, C8).
constexpr float kDilation = 0.3f;
constexpr float kMipDilation = 0.1f;  // GABSPLAT_VARIANT_MIP_FILTER
constexpr float kAlphaMax = 0.99f;
constexpr float kAlphaMin = 1.0f / 255.0f;
constexpr float kTMin = 1e-4f;
constexpr int kTile = GABSPLAT_TILE;
constexpr int kMaxK = GABSPLAT_MAX_K;

// ---- packed gather record (gabsplat_projected.packed), floats -----------------------------------
//  [0..3]   mean2d hi.x, hi.y (fp32 mean, the indexing value), lo.x, lo.y (fp64 residual)
//  [4..7]   L11, L21, L22 (sqrt(log2(e)/2) * Cholesky factor of the conic: G = 2^q, q = -(u^2 + v^2),
//           u = L11 dx + L21 dy, v = L22 dy), qmin = (-ln(255 o) - margin) log2(e)   (envelope reject: skip when q < qmin)
//  [8..11]  opacity, r, g, b
//  [12..]   tail: 2 pi f2D (x,y) * K (radians per pixel), then omega * K; padded to a multiple of 4 floats
__host__ __device__ constexpr int tail_floats(int K) { return 4 * ((3 * K + 3) / 4); }
__host__ __device__ constexpr int packed_floats(int K) { return 12 + tail_floats(K); }

// ---- 2D gradient record accumulated by the blend backward (grad workspace), floats ---------------
//  [0..1] d mean2d   [2..4] S_uu, S_uv, S_vv: the conic's gradient in whitened form (blend_backward.cu)   [5] d opacity   [6..8] d rgb
//  [9..9+2K) d (2 pi f2D) (x,y) * K   [9+2K..9+3K) d omega * K   [9+3K..11+3K) sum |d mean2d| (AbsGS statistic)
//  padded to a multiple of 4 floats
__host__ __device__ constexpr int grad2d_values(int K) { return 11 + 3 * K; }
__host__ __device__ constexpr int grad2d_floats(int K) { return 4 * ((grad2d_values(K) + 3) / 4); }

// ---- blend state saved by the forward for the backward (gabsplat_fwd_out.blend_state) ----------------
// Per half tile h = 2 * tile + warp: counts[h] entries, stored at [2 * list_begin + warp * list_length, ...) of
// ids / masks in the order they were blended (front to back): the primitive id and, for the warp's four
// 16x2 pixel strips, the ballot of the lanes whose pixel blended the primitive.
struct BlendState {
  uint32_t* counts;  // [2 * tiles]
  uint32_t* order;   // [2 * tiles]  half tiles by descending counts (launch order of the backward CTAs)
  uint32_t* ids;     // [2 * capacity]
  uint4* masks;      // [2 * capacity]
};
inline uint64_t blend_state_bytes(uint64_t tiles, uint64_t capacity) {
  const uint64_t a = (2 * tiles * 4 + 255) & ~255ull, o = (2 * tiles * 4 + 255) & ~255ull, b = (2 * capacity * 4 + 255) & ~255ull;
  return a + o + b + 2 * capacity * 16 + 256;
}
inline BlendState make_blend_state(void* p, uint64_t tiles, uint64_t capacity) {
  BlendState s;
  uintptr_t q = ((uintptr_t)p + 255) & ~(uintptr_t)255;
  s.counts = reinterpret_cast<uint32_t*>(q);
  q += (2 * tiles * 4 + 255) & ~255ull;
  s.order = reinterpret_cast<uint32_t*>(q);
  q += (2 * tiles * 4 + 255) & ~255ull;
  s.ids = reinterpret_cast<uint32_t*>(q);
  q += (2 * capacity * 4 + 255) & ~255ull;
  s.masks = reinterpret_cast<uint4*>(q);
  return s;
}

struct Camera {  // device copy of gabsplat_camera plus derived integers
  int width, height, tiles_x, tiles_y;
  float fx, fy, cx, cy;
  float w[12];
  float z_near;
  float bg[3];
};

inline Camera make_camera(const gabsplat_camera& c) {
  Camera k;
  k.width = c.width; k.height = c.height;
  k.tiles_x = (c.width + kTile - 1) / kTile;
  k.tiles_y = (c.height + kTile - 1) / kTile;
  k.fx = c.fx; k.fy = c.fy; k.cx = c.cx; k.cy = c.cy;
  for (int i = 0; i < 12; ++i) k.w[i] = c.world_to_cam[i];
  k.z_near = c.z_near;
  for (int i = 0; i < 3; ++i) k.bg[i] = c.bg[i];
  return k;
}

// ---- optional per-stage device timing (gabsplat_timing_enable / gabsplat_timing_read) -------------
// When enabled, every stage is bracketed by a pair of CUDA events recorded on the stream of the call;
// the records are read back (elapsed ms per stage launch) by gabsplat_timing_read.
struct StageTimer {
  struct Rec { int stage; cudaEvent_t a, b; };
  bool on = false;
  std::vector<cudaEvent_t> pool;
  size_t used = 0;
  std::vector<Rec> recs;
  cudaEvent_t take() {
    if (used == pool.size()) {
      cudaEvent_t e = nullptr;
      cudaEventCreate(&e);
      pool.push_back(e);
    }
    return pool[used++];
  }
  void begin(int stage, cudaStream_t st) {
    if (!on) return;
    Rec r{stage, take(), take()};
    cudaEventRecord(r.a, st);
    recs.push_back(r);
  }
  void end(cudaStream_t st) {
    if (!on || recs.empty()) return;
    cudaEventRecord(recs.back().b, st);
  }
  void reset() { recs.clear(); used = 0; }
  void destroy() {
    for (cudaEvent_t e : pool) cudaEventDestroy(e);
    pool.clear();
    reset();
  }
};

// ---- programmatic dependent launch ---------------------------------------------------------------------
// The small kernels of a call form a chain of dependent launches whose cost is mostly launch latency.  Launched
// with launch_pdl, a kernel may be scheduled while its predecessor in the stream drains; it must call pdl_wait()
// before it touches anything the predecessor wrote (first statement of every kernel launched this way).
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
#endif
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// SMs of the current device, for the grid-stride kernels whose grids are a multiple of it (148 on B200); looked up once
// per device ordinal.
inline int sm_count() {
  static std::atomic<int> cached[64];
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  int n = cached[dev].load(std::memory_order_relaxed);
  if (n == 0) {
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    cached[dev].store(n, std::memory_order_relaxed);
  }
  return n;
}

// Number of kernels launched by this library since it was loaded (gabsplat_kernel_launches).
extern std::atomic<unsigned long long> g_kernel_launches;
inline void launched(int n = 1) { g_kernel_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

// ---- launchers (one per .cu file); each returns the cudaError_t of its last launch ---------------
cudaError_t launch_preprocess(const gabsplat_scene& s, const Camera& cam, const gabsplat_projected& out,
                              cudaStream_t st, cudaStream_t value_stream, cudaEvent_t index_done);
cudaError_t launch_bin_sort(int N, const gabsplat_projected& proj, const Camera& cam, const gabsplat_binning& bin,
                            StageTimer& tm, int place_bands, cudaStream_t st);
cudaError_t launch_blend_forward(int K, const Camera& cam, const gabsplat_projected& proj,
                                 const gabsplat_binning& bin, const gabsplat_fwd_out& out, const BlendState* save,
                                 cudaStream_t st);
cudaError_t launch_blend_aux(int N, int K, const float* weights, const Camera& cam, const gabsplat_projected& proj,
                             const gabsplat_binning& bin, float4* aux, float* image, float* final_T, uint32_t* n_contrib,
                             cudaStream_t st);
cudaError_t launch_count_pairs(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                               uint32_t* counters, cudaStream_t st);
cudaError_t launch_blend_backward(int N, int K, bool want_abs, const Camera& cam, const gabsplat_projected& proj,
                                  const gabsplat_binning& bin, const gabsplat_fwd_out& fwd, const BlendState& saved,
                                  const float* dL_dimage, float* grad2d, cudaStream_t st);
cudaError_t launch_grad_zero(const gabsplat_scene& s, const gabsplat_grads& g, cudaStream_t st);
cudaError_t launch_preprocess_backward(const gabsplat_scene& s, const Camera& cam, const gabsplat_projected& proj,
                                       const gabsplat_binning& bin, float* grad2d, const gabsplat_grads& g, cudaStream_t st);
// the depth-ordered ids of the visible primitives and their number, as gabsplat_bin_sort left them in bin.workspace
void binning_visible_list(const gabsplat_binning& bin, int N, int ntiles, const uint32_t** order, const uint32_t** n_vis);

// order[] = the tiles by descending work, work(t) = pairs[t].y - pairs[t].x (sum == false) or pairs[t].x + pairs[t].y
cudaError_t launch_tile_order(const uint32_t* pairs, bool sum, int ntiles, uint32_t* order, cudaStream_t st);
// order[] = the items 0..n-1 by descending work[item]
cudaError_t launch_half_tile_order(const uint32_t* work, int n, uint32_t* order, cudaStream_t st);

uint64_t loss_workspace_bytes(int W, int H);
cudaError_t launch_loss(int W, int H, const float* image, const float* target, float lambda, float* loss_out,
                        float* dL_dimage, void* workspace, cudaStream_t st);

// instrumentation (blend_forward.cu, peaks.cu)
cudaError_t launch_trace_pixels(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin, int n,
                                const int32_t* pixels, const uint32_t* offsets, uint32_t* entries, float* colour_T,
                                uint32_t* info, cudaStream_t st);
cudaError_t launch_probe_sincos(int n, const float* phase, float* c, float* s, cudaStream_t st);
cudaError_t measure_peaks(float* results_host, void* scratch, cudaStream_t st);

// argument checks of the ABI (api.cu): the INVALID_ARG conditions of gabsplat.h on a camera / a scene of device or host pointers
bool camera_ok(const gabsplat_camera* c);
bool scene_ok(const gabsplat_scene* s);

uint64_t sort_workspace_bytes(int N, uint64_t capacity, int ntiles);
bool keys_optional(int ntiles);  // true when the binning never reads gabsplat_binning.keys itself

}  // namespace gabsplat

// The context (opaque to callers).  It owns no per-call state: a pinned readback slot, a side stream for work that has
// no consumer on the critical path, two copy streams for gabsplat_render_host, and the events that order them.
struct gabsplat_ctx {
  int device;
  uint64_t* pinned_count;  // 8-byte pinned readback slot for D
  cudaStream_t side;       // side stream: the zeroing of the gradient arrays overlaps the blend backward
  cudaEvent_t ev_fork, ev_join;
  cudaStream_t copy_in, copy_out;            // gabsplat_render_host: uploads / downloads beside the kernels
  cudaEvent_t ev_copy[5];                    // ... and their ordering
  void* scratch;           // 256 bytes of device scratch (instrumentation)
  int place_bands;         // 0 = automatic (gabsplat_set_place_bands)
  gabsplat::StageTimer timer;
  char error[256];
};

// S1 + S2 as gabsplat_preprocess_bin_sort runs them; `value_inputs_ready` (may be null) is an event the fp64 value track
// waits for on the side stream: gabsplat_render_host starts the indexing track and the binning as soon as means, scales
// and rotations have arrived, while the rest of the scene is still on its way.
int32_t gabsplat_preprocess_bin_sort_ordered(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                             gabsplat_projected* proj, gabsplat_binning* bin, uint64_t* num_instances_host,
                                             void* stream, cudaEvent_t value_inputs_ready);
