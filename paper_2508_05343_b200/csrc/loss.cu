// the training loss of PAPER.md:171 Eq.14 on the device, forward and backward,
//     L = (1 - lambda) L1 + lambda (1 - mean SSIM),
// SSIM per channel with the 11x11 Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2 of [25]
// (reading C25).  It produces dL/dimage, the input of gabsplat_render_backward, without leaving the GPU.
//
// Two tiled passes, both HBM bound (26 MB in + 39 MB out, then 65 MB in + 13 MB out at 1297x840):
//   ssim_maps_kernel   per 32x16 tile of one channel: the four windowed sums w*x, w*y, w*(x^2 + y^2), w*xy (SSIM needs
//                      the two second moments only through their sum) as a
//                      separable 11-tap filter through shared memory, SSIM and its three partial derivatives
//                      (dS/dmx, dS/dExx, dS/dExy) per pixel, per-CTA partial sums of |x - y| and SSIM
//   loss_grad_kernel   the same separable filter over the three derivative maps, combined with x, y and sign(x - y)
// The windowed sums are accumulated in fp64 (Exx - mx^2 cancels against C2 = 9e-4) and the partial sums are reduced in
// a fixed order, so the loss is deterministic.  What the kernels spend is the fp64 filter arithmetic (11 + 11 DFMA per
// quantity and pixel, plus the halo rows), so everything around it is kept off the instruction stream: a thread of
// the horizontal pass converts and multiplies each input ONCE and feeds it to the 4 neighbouring outputs it owns; a
// thread of the vertical pass owns two adjacent rows, whose 11-row windows share 10 rows.
#include <mutex>

#include "common.cuh"

namespace gabsplat {
namespace {

constexpr int kR = 5;             // window radius
constexpr int kTX = 32, kTY = 16;  // output tile: two pixels per thread (rows 2 ty and 2 ty + 1)
constexpr int kHX = kTX + 2 * kR, kHY = kTY + 2 * kR;
constexpr int kLossThreads = 256;
constexpr double kC1 = 0.01 * 0.01, kC2 = 0.03 * 0.03;

struct Taps { double g[2 * kR + 1]; };

inline Taps make_taps() {
  Taps t;
  double sum = 0.0;
  for (int i = 0; i <= 2 * kR; ++i) { t.g[i] = exp(-(double)((i - kR) * (i - kR)) / (2.0 * 1.5 * 1.5)); sum += t.g[i]; }
  for (int i = 0; i <= 2 * kR; ++i) t.g[i] /= sum;
  return t;
}

// Separable filter of NQ quantities over one tile.  in(r, c, v) gives the NQ input values at halo position (r, c)
// (zero outside the image); s_h[q][kHY][kTX] receives the horizontal sums; out[q][h] = the filtered value at the
// thread's output pixels (tile rows 2 ty + h, column tx).  Every sum adds its 11 terms in tap order.
constexpr int kGroup = 4;                     // horizontal pass: adjacent outputs per thread
constexpr int kGroupsPerRow = kTX / kGroup;
template <int NQ, typename In>
__device__ __forceinline__ void separable(const Taps& taps, In in, double (*s_h)[kHY][kTX], int tx, int ty, double (&out)[NQ][2]) {
  if (threadIdx.x < kHY * kGroupsPerRow) {
    const int r = threadIdx.x / kGroupsPerRow, c0 = kGroup * (threadIdx.x - r * kGroupsPerRow);
    double acc[kGroup][NQ];
#pragma unroll
    for (int o = 0; o < kGroup; ++o)
#pragma unroll
      for (int q = 0; q < NQ; ++q) acc[o][q] = 0.0;
#pragma unroll
    for (int j = 0; j < kGroup + 2 * kR; ++j) {
      double v[NQ];
      in(r, c0 + j, v);
#pragma unroll
      for (int o = 0; o < kGroup; ++o) {
        if (j - o >= 0 && j - o <= 2 * kR) {
#pragma unroll
          for (int q = 0; q < NQ; ++q) acc[o][q] += taps.g[j - o] * v[q];
        }
      }
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q)
#pragma unroll
      for (int o = 0; o < kGroup; ++o) s_h[q][r][c0 + o] = acc[o][q];
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < NQ; ++q) {
    double a0 = 0.0, a1 = 0.0;
#pragma unroll
    for (int i = 0; i <= 2 * kR + 1; ++i) {
      const double v = s_h[q][2 * ty + i][tx];
      if (i <= 2 * kR) a0 += taps.g[i] * v;
      if (i >= 1) a1 += taps.g[i - 1] * v;
    }
    out[q][0] = a0;
    out[q][1] = a1;
  }
}

// the (kHY x kHX) halo of one channel of NI images -> shared memory (zero outside the image): a warp per row
template <int NI>
__device__ __forceinline__ void load_halo(int W, int H, int x0, int y0, const float* const (&src)[NI], float (*const (&dst)[NI])[kHX]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int r = warp; r < kHY; r += kLossThreads / 32) {
    const int gy = y0 + r;
    const bool row_in = gy >= 0 && gy < H;
    const size_t base = (size_t)gy * W;
    for (int c = lane; c < kHX; c += 32) {
      const int gx = x0 + c;
      const bool ok = row_in && gx >= 0 && gx < W;
#pragma unroll
      for (int i = 0; i < NI; ++i) dst[i][r][c] = ok ? __ldg(src[i] + base + gx) : 0.f;
    }
  }
}

__global__ void __launch_bounds__(kLossThreads, 4) ssim_maps_kernel(int W, int H, Taps taps, const float* __restrict__ image,
                                                                const float* __restrict__ target, float* __restrict__ maps,
                                                                double* __restrict__ partials) {
  __shared__ float s_x[kHY][kHX], s_y[kHY][kHX];
  __shared__ double s_h[4][kHY][kTX];
  __shared__ double s_red[2][kLossThreads / 32];
  const int ch = blockIdx.z;
  const size_t HW = (size_t)W * H;
  const float* x = image + ch * HW;
  const float* y = target + ch * HW;
  const int x0 = blockIdx.x * kTX - kR, y0 = blockIdx.y * kTY - kR;
  {
    const float* const src[2] = {x, y};
    float (*const dst[2])[kHX] = {s_x, s_y};
    load_halo<2>(W, H, x0, y0, src, dst);
  }
  __syncthreads();
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  double f[4][2];
  separable<4>(taps, [&](int r, int c, double (&v)[4]) {
    const double a = s_x[r][c], b = s_y[r][c];
    v[0] = a; v[1] = b; v[2] = a * a + b * b; v[3] = a * b;
  }, s_h, tx, ty, f);
  double sum_l1 = 0.0, sum_s = 0.0;
  const int gx = blockIdx.x * kTX + tx;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int gy = blockIdx.y * kTY + 2 * ty + h;
    if (gx >= W || gy >= H) continue;
    const double mx = f[0][h], my = f[1][h], exx_eyy = f[2][h], exy = f[3][h];
    const double a1 = 2.0 * mx * my + kC1, a2 = 2.0 * (exy - mx * my) + kC2;
    const double b1 = mx * mx + my * my + kC1, b2 = exx_eyy - (mx * mx + my * my) + kC2;
    const double ib = 1.0 / (b1 * b2);
    const double sv = a1 * a2 * ib;
    const size_t p = (size_t)gy * W + gx;
    maps[(0 * 3 + ch) * HW + p] = (float)((2.0 * my * a2 - 2.0 * my * a1) * ib - sv * (2.0 * mx / b1 - 2.0 * mx / b2));
    maps[(1 * 3 + ch) * HW + p] = (float)(-sv / b2);
    maps[(2 * 3 + ch) * HW + p] = (float)(2.0 * a1 * ib);
    sum_s += sv;
    sum_l1 += fabs((double)s_x[2 * ty + h + kR][tx + kR] - (double)s_y[2 * ty + h + kR][tx + kR]);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    sum_l1 += __shfl_xor_sync(0xffffffffu, sum_l1, d);
    sum_s += __shfl_xor_sync(0xffffffffu, sum_s, d);
  }
  if (tx == 0) { s_red[0][ty] = sum_l1; s_red[1][ty] = sum_s; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int w = 0; w < kLossThreads / 32; ++w) { a += s_red[0][w]; b += s_red[1][w]; }
    const size_t blk = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    partials[2 * blk] = a;
    partials[2 * blk + 1] = b;
  }
}

// one CTA: the partial sums in index order -> (L, L1, mean SSIM)
__global__ void __launch_bounds__(256) loss_reduce_kernel(const double* __restrict__ partials, int nblocks, double n, float lambda,
                                                          float* __restrict__ loss_out) {
  __shared__ double s_a[256], s_b[256];
  double a = 0.0, b = 0.0;
  const int per = (nblocks + 255) / 256;
  for (int j = threadIdx.x * per; j < min(nblocks, (int)(threadIdx.x + 1) * per); ++j) { a += partials[2 * j]; b += partials[2 * j + 1]; }
  s_a[threadIdx.x] = a; s_b[threadIdx.x] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
    double ta = 0.0, tb = 0.0;
    for (int j = 0; j < 256; ++j) { ta += s_a[j]; tb += s_b[j]; }
    const double l1 = ta / n, ssim = tb / n;
    loss_out[0] = (float)((1.0 - (double)lambda) * l1 + (double)lambda * (1.0 - ssim));
    loss_out[1] = (float)l1;
    loss_out[2] = (float)ssim;
  }
}

__global__ void __launch_bounds__(kLossThreads) loss_grad_kernel(int W, int H, Taps taps, const float* __restrict__ image,
                                                                const float* __restrict__ target, const float* __restrict__ maps,
                                                                float lambda, float* __restrict__ dL_dimage) {
  __shared__ float s_in[3][kHY][kHX];
  __shared__ double s_h[3][kHY][kTX];
  const int ch = blockIdx.z;
  const size_t HW = (size_t)W * H;
  const int x0 = blockIdx.x * kTX - kR, y0 = blockIdx.y * kTY - kR;
  {
    const float* const src[3] = {maps + (0 * 3 + ch) * HW, maps + (1 * 3 + ch) * HW, maps + (2 * 3 + ch) * HW};
    float (*const dst[3])[kHX] = {s_in[0], s_in[1], s_in[2]};
    load_halo<3>(W, H, x0, y0, src, dst);
  }
  __syncthreads();
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  double f[3][2];
  separable<3>(taps, [&](int r, int c, double (&v)[3]) {
    v[0] = s_in[0][r][c]; v[1] = s_in[1][r][c]; v[2] = s_in[2][r][c];
  }, s_h, tx, ty, f);
  const double n = 3.0 * (double)HW;
  const double gs = -(double)lambda / n, g1 = (1.0 - (double)lambda) / n;
  const int gx = blockIdx.x * kTX + tx;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int gy = blockIdx.y * kTY + 2 * ty + h;
    if (gx >= W || gy >= H) continue;
    const size_t p = (size_t)gy * W + gx;
    const double xv = image[ch * HW + p], yv = target[ch * HW + p];
    const double d = xv - yv;
    const double sgn = d > 0.0 ? 1.0 : (d < 0.0 ? -1.0 : 0.0);
    dL_dimage[ch * HW + p] = (float)(gs * (f[0][h] + 2.0 * xv * f[1][h] + yv * f[2][h]) + g1 * sgn);
  }
}

}  // namespace

uint64_t loss_workspace_bytes(int W, int H) {
  const uint64_t hw = (uint64_t)W * H;
  const uint64_t blocks = (uint64_t)((W + kTX - 1) / kTX) * ((H + kTY - 1) / kTY) * 3;
  return 9 * hw * sizeof(float) + 256 + blocks * 2 * sizeof(double) + 256;
}

cudaError_t launch_loss(int W, int H, const float* image, const float* target, float lambda, float* loss_out,
                        float* dL_dimage, void* workspace, cudaStream_t st) {
  static const Taps taps = make_taps();
  const uint64_t hw = (uint64_t)W * H;
  float* maps = reinterpret_cast<float*>(((uintptr_t)workspace + 255) & ~(uintptr_t)255);
  double* partials = reinterpret_cast<double*>(((uintptr_t)(maps + 9 * hw) + 255) & ~(uintptr_t)255);
  const dim3 grid((W + kTX - 1) / kTX, (H + kTY - 1) / kTY, 3);
  ssim_maps_kernel<<<grid, kLossThreads, 0, st>>>(W, H, taps, image, target, maps, partials);
  loss_reduce_kernel<<<1, 256, 0, st>>>(partials, (int)(grid.x * grid.y * grid.z), 3.0 * (double)hw, lambda, loss_out);
  launched(2);
  if (dL_dimage) {
    loss_grad_kernel<<<grid, kLossThreads, 0, st>>>(W, H, taps, image, target, maps, lambda, dL_dimage);
    launched();
  }
  return cudaGetLastError();
}

}  // namespace gabsplat

// ---- gabsplat_loss_static: the same loss for callers that have no way to obtain device scratch ----------------
//
// gabsplat_loss needs a workspace (the nine derivative maps between its two passes and the per-CTA partial sums),
// and the workspace has to come from somewhere: cudaMalloc, or a framework allocator sitting on top of it.  Some
// callers cannot do that.  A plugin running inside someone else's engine is handed its input and output buffers
// and nothing else; a real-time or safety-reviewed loop is forbidden to touch the allocator after start-up
// (cudaMalloc takes a process-wide lock and may synchronise the device); a caller on a memory-capped GPU may find
// the pool exhausted or fragmented at the moment it asks.  For them the scratch lives in the library image itself:
// a file-scope __device__ array that the CUDA runtime places on every GPU that loads this module and that stays there
// until the process exits.  Nothing is allocated or freed by this entry point, ever.
//
// The price is a fixed ceiling (kStaticMaxPixels, below) and a single shared copy per GPU: see the header.
namespace gabsplat {
namespace {

constexpr int kStaticMaxPixels = 512 * 512;  // width * height; 36 bytes of maps per pixel -> 9 MiB
constexpr int kStaticMaxSide = 2048;         // bounds the CTA count of a thin strip: 3 (W/32 + 1)(H/16 + 1) <= 3 * 705
constexpr int kStaticMaxBlocks = 3 * 768;
constexpr size_t kStaticMapsBytes = (size_t)9 * kStaticMaxPixels * sizeof(float);  // a multiple of 256
constexpr size_t kStaticBytes = kStaticMapsBytes + (size_t)kStaticMaxBlocks * 2 * sizeof(double);
static_assert(kStaticMapsBytes % 256 == 0, "the partial sums follow the maps and hold doubles");

// The scratch itself.  In HOST code this name is only a handle the runtime recognises -- it is not a device address,
// and handing it to a kernel would make the kernel write through a host pointer.  The address the kernels may use
// comes from cudaGetSymbolAddress (static_scratch below) and differs from GPU to GPU.
static __device__ __align__(256) unsigned char g_loss_scratch[kStaticBytes];

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned char* g_static_address[kStaticMaxDevices] = {};  // per device ordinal; resolved on the first call there
thread_local const char* t_static_error = "no error";

// Device address of g_loss_scratch on the CURRENT device, looked up once per device.  The look-up may make the
// runtime load this module onto the device, which is why the first call on a device belongs before any capture.
cudaError_t static_scratch(unsigned char** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_address[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_loss_scratch);
    if (e != cudaSuccess) return e;
    g_static_address[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_static_address[dev];
  return cudaSuccess;
}

}  // namespace
}  // namespace gabsplat

extern "C" uint64_t gabsplat_loss_static_max_pixels(void) { return (uint64_t)gabsplat::kStaticMaxPixels; }

extern "C" const char* gabsplat_loss_static_last_error(void) { return gabsplat::t_static_error; }

extern "C" int32_t gabsplat_loss_static(int32_t width, int32_t height, const float* image, const float* target, float lambda,
                                        float* loss_out, float* dL_dimage, void* stream) {
  using namespace gabsplat;
  if (width <= 0 || height <= 0 || !image || !target || !loss_out || !(lambda >= 0.f && lambda <= 1.f)) {
    t_static_error = "loss_static: bad size, lambda or null pointer";
    return GABSPLAT_INVALID_ARG;
  }
  const dim3 grid((width + kTX - 1) / kTX, (height + kTY - 1) / kTY, 3);
  if (width > kStaticMaxSide || height > kStaticMaxSide || (int64_t)width * height > (int64_t)kStaticMaxPixels ||
      (uint64_t)grid.x * grid.y * grid.z > (uint64_t)kStaticMaxBlocks) {
    t_static_error = "loss_static: image larger than the built-in scratch (width * height <= 262144, each side <= 2048); "
                     "use gabsplat_loss with a caller-provided workspace";
    return GABSPLAT_CAPACITY;
  }
  unsigned char* scratch = nullptr;
  cudaError_t e = static_scratch(&scratch);
  if (e != cudaSuccess) {
    t_static_error = cudaGetErrorString(e);
    return GABSPLAT_CUDA;
  }
  // Every map value and partial sum that is read below is written first by this same call, so the previous call's
  // leftovers in the array need no clearing.
  float* maps = reinterpret_cast<float*>(scratch);
  double* partials = reinterpret_cast<double*>(scratch + kStaticMapsBytes);
  static const Taps taps = make_taps();
  const cudaStream_t st = (cudaStream_t)stream;
  const uint64_t hw = (uint64_t)width * height;
  ssim_maps_kernel<<<grid, kLossThreads, 0, st>>>(width, height, taps, image, target, maps, partials);
  loss_reduce_kernel<<<1, 256, 0, st>>>(partials, (int)(grid.x * grid.y * grid.z), 3.0 * (double)hw, lambda, loss_out);
  launched(2);
  if (dL_dimage) {
    loss_grad_kernel<<<grid, kLossThreads, 0, st>>>(width, height, taps, image, target, maps, lambda, dL_dimage);
    launched();
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    t_static_error = cudaGetErrorString(e);
    return GABSPLAT_CUDA;
  }
  return GABSPLAT_OK;
}
