// the training loss of PAPER.md:171 Eq.14 on the device, forward and backward,
//     L = (1 - lambda) L1 + lambda (1 - mean SSIM),
// SSIM per channel with the 11x11 Gaussian window (sigma 1.5), zero padding, C1 = 0.01^2, C2 = 0.03^2 of [25]
// (reading C25).  It produces dL/dimage, the input of gabsplat_render_backward, without leaving the GPU.
//
// Two tiled passes, both HBM bound (26 MB in + 39 MB out, then 65 MB in + 13 MB out at 1297x840):
//   ssim_maps_kernel   per 32x16 tile of one channel: the five windowed sums w*x, w*y, w*x^2, w*y^2, w*xy as a
//                      separable 11-tap filter through shared memory, SSIM and its three partial derivatives
//                      (dS/dmx, dS/dExx, dS/dExy) per pixel, per-CTA partial sums of |x - y| and SSIM
//   loss_grad_kernel   the same separable filter over the three derivative maps, combined with x, y and sign(x - y)
// The windowed sums are accumulated in fp64 (Exx - mx^2 cancels against C2 = 9e-4; the arithmetic is free next to
// the memory traffic) and the partial sums are reduced in a fixed order, so the loss is deterministic.
#include "common.cuh"

namespace gabsplat {
namespace {

constexpr int kR = 5;             // window radius
constexpr int kTX = 32, kTY = 16;  // output tile: two pixels per thread (rows ty and ty + 8)
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
// thread's output pixels (tile rows ty + 8 h, column tx).
template <int NQ, typename In>
__device__ __forceinline__ void separable(const Taps& taps, In in, double (*s_h)[kHY][kTX], int tx, int ty, double (&out)[NQ][2]) {
  for (int e = threadIdx.x; e < kHY * kTX; e += kLossThreads) {
    const int r = e / kTX, c = e - r * kTX;
    double acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
#pragma unroll
    for (int j = 0; j <= 2 * kR; ++j) {
      double v[NQ];
      in(r, c + j, v);
#pragma unroll
      for (int q = 0; q < NQ; ++q) acc[q] += taps.g[j] * v[q];
    }
#pragma unroll
    for (int q = 0; q < NQ; ++q) s_h[q][r][c] = acc[q];
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      double acc = 0.0;
#pragma unroll
      for (int i = 0; i <= 2 * kR; ++i) acc += taps.g[i] * s_h[q][ty + 8 * h + i][tx];
      out[q][h] = acc;
    }
}

__global__ void __launch_bounds__(kLossThreads) ssim_maps_kernel(int W, int H, Taps taps, const float* __restrict__ image,
                                                                const float* __restrict__ target, float* __restrict__ maps,
                                                                double* __restrict__ partials) {
  __shared__ float s_x[kHY][kHX], s_y[kHY][kHX];
  __shared__ double s_h[5][kHY][kTX];
  __shared__ double s_red[2][kLossThreads / 32];
  const int ch = blockIdx.z;
  const size_t HW = (size_t)W * H;
  const float* x = image + ch * HW;
  const float* y = target + ch * HW;
  const int x0 = blockIdx.x * kTX - kR, y0 = blockIdx.y * kTY - kR;
  for (int e = threadIdx.x; e < kHY * kHX; e += kLossThreads) {
    const int r = e / kHX, c = e - r * kHX;
    const int gx = x0 + c, gy = y0 + r;
    const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
    s_x[r][c] = in ? x[(size_t)gy * W + gx] : 0.f;
    s_y[r][c] = in ? y[(size_t)gy * W + gx] : 0.f;
  }
  __syncthreads();
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  double f[5][2];
  separable<5>(taps, [&](int r, int c, double (&v)[5]) {
    const double a = s_x[r][c], b = s_y[r][c];
    v[0] = a; v[1] = b; v[2] = a * a; v[3] = b * b; v[4] = a * b;
  }, s_h, tx, ty, f);
  double sum_l1 = 0.0, sum_s = 0.0;
  const int gx = blockIdx.x * kTX + tx;
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int gy = blockIdx.y * kTY + ty + 8 * h;
    if (gx >= W || gy >= H) continue;
    const double mx = f[0][h], my = f[1][h], exx = f[2][h], eyy = f[3][h], exy = f[4][h];
    const double a1 = 2.0 * mx * my + kC1, a2 = 2.0 * (exy - mx * my) + kC2;
    const double b1 = mx * mx + my * my + kC1, b2 = (exx - mx * mx) + (eyy - my * my) + kC2;
    const double ib = 1.0 / (b1 * b2);
    const double sv = a1 * a2 * ib;
    const size_t p = (size_t)gy * W + gx;
    maps[(0 * 3 + ch) * HW + p] = (float)((2.0 * my * a2 - 2.0 * my * a1) * ib - sv * (2.0 * mx / b1 - 2.0 * mx / b2));
    maps[(1 * 3 + ch) * HW + p] = (float)(-sv / b2);
    maps[(2 * 3 + ch) * HW + p] = (float)(2.0 * a1 * ib);
    sum_s += sv;
    sum_l1 += fabs((double)s_x[ty + 8 * h + kR][tx + kR] - (double)s_y[ty + 8 * h + kR][tx + kR]);
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
  for (int e = threadIdx.x; e < kHY * kHX; e += kLossThreads) {
    const int r = e / kHX, c = e - r * kHX;
    const int gx = x0 + c, gy = y0 + r;
    const bool in = gx >= 0 && gx < W && gy >= 0 && gy < H;
    const size_t p = (size_t)gy * W + gx;
#pragma unroll
    for (int q = 0; q < 3; ++q) s_in[q][r][c] = in ? maps[(q * 3 + ch) * HW + p] : 0.f;
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
    const int gy = blockIdx.y * kTY + ty + 8 * h;
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
