// S1 / K1: projection of every primitive to the image plane.
//   Sigma' = J W Sigma W^T J^T (Eq.2), conic of the dilated 2x2 block (Eq.3 :101),
//   f2D_k = Eq.9-11 (:145, :414, :150-154) in the closed form U^-1 T Sigma f_k (reading C2),
//   mu2D (:99), radius / tile rectangle / tiles_touched, SH colour (:83).
//
// Two arithmetic tracks per primitive:
//   * the INDEXING track -- visibility, depth key, radius, rectangle -- is the normative fp32 operation
//     sequence of DESIGN.md ("Normative fp32 sequence"), written with round-to-nearest intrinsics so that no
//     compiler flag can fuse or reorder it: it must agree bit for bit with any IEEE-754 implementation of it;
//   * the VALUE track -- conic, f2D, colour, sub-pixel mean -- is evaluated in fp64 and rounded once to fp32
//     for storage (the kernel is HBM-bound: ~150 k visible primitives x a few hundred flops is free, and it
//     keeps ill-conditioned covariances, whose 2x2 inverse loses cond(U) digits in fp32, inside the 1e-4 bar).
#include "common.cuh"
#include "sh.cuh"

namespace gabsplat {
namespace {

__device__ __forceinline__ float fmul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float fadd(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float fsub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float ffma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float fdiv(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float fsqrt(float a) { return __fsqrt_rn(a); }
__device__ __forceinline__ float fclamp(float v, float lo, float hi) { return fminf(fmaxf(v, lo), hi); }

struct Index {  // result of the indexing track
  bool visible;
  float depth, m2x, m2y;
  int radius, x0, y0, x1, y1;
  uint32_t tiles;
};

__device__ Index index_track(const Camera& c, float dilation, float mx, float my, float mz, const float* __restrict__ sc,
                             const float* __restrict__ q) {
  Index o;
  o.visible = false; o.tiles = 0; o.radius = 0; o.x0 = o.y0 = o.x1 = o.y1 = 0; o.depth = o.m2x = o.m2y = 0.f;
  float t[3];
#pragma unroll
  for (int a = 0; a < 3; ++a)
    t[a] = ffma(c.w[4 * a], mx, ffma(c.w[4 * a + 1], my, ffma(c.w[4 * a + 2], mz, c.w[4 * a + 3])));
  if (!(t[2] > c.z_near)) return o;
  const float qw = q[0], qx = q[1], qy = q[2], qz = q[3];
  float R[3][3];
  R[0][0] = fsub(1.0f, fmul(2.0f, fadd(fmul(qy, qy), fmul(qz, qz))));
  R[0][1] = fmul(2.0f, fsub(fmul(qx, qy), fmul(qw, qz)));
  R[0][2] = fmul(2.0f, fadd(fmul(qx, qz), fmul(qw, qy)));
  R[1][0] = fmul(2.0f, fadd(fmul(qx, qy), fmul(qw, qz)));
  R[1][1] = fsub(1.0f, fmul(2.0f, fadd(fmul(qx, qx), fmul(qz, qz))));
  R[1][2] = fmul(2.0f, fsub(fmul(qy, qz), fmul(qw, qx)));
  R[2][0] = fmul(2.0f, fsub(fmul(qx, qz), fmul(qw, qy)));
  R[2][1] = fmul(2.0f, fadd(fmul(qy, qz), fmul(qw, qx)));
  R[2][2] = fsub(1.0f, fmul(2.0f, fadd(fmul(qx, qx), fmul(qy, qy))));
  float M[3][3], Sg[3][3];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) M[a][b] = fmul(R[a][b], sc[b]);
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) Sg[a][b] = ffma(M[a][2], M[b][2], ffma(M[a][1], M[b][1], fmul(M[a][0], M[b][0])));
  const float limx = fmul(1.3f, fdiv(fmul(0.5f, (float)c.width), c.fx));
  const float limy = fmul(1.3f, fdiv(fmul(0.5f, (float)c.height), c.fy));
  const float rx = fdiv(t[0], t[2]), ry = fdiv(t[1], t[2]);
  const float ux = fclamp(rx, -limx, limx), uy = fclamp(ry, -limy, limy);
  const float J00 = fdiv(c.fx, t[2]), J11 = fdiv(c.fy, t[2]);
  const float J02 = -fmul(J00, ux), J12 = -fmul(J11, uy);
  float T[2][3], V[2][3];
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    T[0][b] = ffma(J02, c.w[8 + b], fmul(J00, c.w[b]));
    T[1][b] = ffma(J12, c.w[8 + b], fmul(J11, c.w[4 + b]));
  }
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) V[a][b] = ffma(T[a][2], Sg[2][b], ffma(T[a][1], Sg[1][b], fmul(T[a][0], Sg[0][b])));
  const float U00 = ffma(V[0][2], T[0][2], ffma(V[0][1], T[0][1], fmul(V[0][0], T[0][0])));
  const float U01 = ffma(V[0][2], T[1][2], ffma(V[0][1], T[1][1], fmul(V[0][0], T[1][0])));
  const float U11 = ffma(V[1][2], T[1][2], ffma(V[1][1], T[1][1], fmul(V[1][0], T[1][0])));
  const float A = fadd(U00, dilation), C = fadd(U11, dilation);
  const float det = fsub(fmul(A, C), fmul(U01, U01));
  if (!(det > 0.0f)) return o;
  const float mid = fmul(0.5f, fadd(A, C)), hd = fmul(0.5f, fsub(A, C));
  const float lam = fadd(mid, fsqrt(ffma(hd, hd, fmul(U01, U01))));
  const float rf = ceilf(fmul(3.0f, fsqrt(lam)));
  const float m2x = ffma(c.fx, rx, c.cx), m2y = ffma(c.fy, ry, c.cy);
  const float gxf = (float)c.tiles_x, gyf = (float)c.tiles_y;
  o.x0 = (int)fclamp(fmul(fsub(m2x, rf), 0.0625f), 0.0f, gxf);
  o.y0 = (int)fclamp(fmul(fsub(m2y, rf), 0.0625f), 0.0f, gyf);
  o.x1 = (int)fclamp(fmul(fadd(fadd(m2x, rf), 15.0f), 0.0625f), 0.0f, gxf);
  o.y1 = (int)fclamp(fmul(fadd(fadd(m2y, rf), 15.0f), 0.0625f), 0.0f, gyf);
  const int area = (o.x1 - o.x0) * (o.y1 - o.y0);
  if (area <= 0) return o;
  o.visible = true;
  o.tiles = (uint32_t)area;
  o.radius = (int)rf;
  o.depth = t[2];
  o.m2x = m2x; o.m2y = m2y;
  return o;
}

// fp64 value track of one visible primitive; everything it stores is rounded once to fp32.
// VARIANT: compiled with the primitive variants of gabsplat_scene.variant (f4); the plain instantiation carries none of
// their registers
template <bool VARIANT>
__device__ __forceinline__ void value_track(const gabsplat_scene& s, const Camera& c, const gabsplat_projected& out,
                                            const int i) {
  // the fp32 mean of the indexing track (index_kernel wrote it): the packed record carries it with its fp64 residual
  const float2 m2 = reinterpret_cast<const float2*>(out.mean2d)[i];
  const int K = s.K;
  const float mx = s.means[3 * i], my = s.means[3 * i + 1], mz = s.means[3 * i + 2];
  float sc[3], q[4];
#pragma unroll
  for (int a = 0; a < 3; ++a) sc[a] = s.scales[3 * i + a];
  {
    const float4 qv = reinterpret_cast<const float4*>(s.rotations)[i];
    q[0] = qv.x; q[1] = qv.y; q[2] = qv.z; q[3] = qv.w;
  }
  // ---------------- value track (fp64) ----------------
  double Wm[3][3], tau[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int b = 0; b < 3; ++b) Wm[a][b] = (double)c.w[4 * a + b];
    tau[a] = (double)c.w[4 * a + 3];
  }
  const double mu[3] = {(double)mx, (double)my, (double)mz};
  double t[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) t[a] = Wm[a][0] * mu[0] + Wm[a][1] * mu[1] + Wm[a][2] * mu[2] + tau[a];
  const double tz = t[2];
  // Sigma = R diag(s^2) R^T
  double Sg[3][3], R[3][3];
  const double s2[3] = {(double)sc[0] * sc[0], (double)sc[1] * sc[1], (double)sc[2] * sc[2]};
  {
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0][0] = 1 - 2 * (y * y + z * z); R[0][1] = 2 * (x * y - w * z); R[0][2] = 2 * (x * z + w * y);
    R[1][0] = 2 * (x * y + w * z); R[1][1] = 1 - 2 * (x * x + z * z); R[1][2] = 2 * (y * z - w * x);
    R[2][0] = 2 * (x * z - w * y); R[2][1] = 2 * (y * z + w * x); R[2][2] = 1 - 2 * (x * x + y * y);
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) Sg[a][b] = R[a][0] * s2[0] * R[b][0] + R[a][1] * s2[1] * R[b][1] + R[a][2] * s2[2] * R[b][2];
  }
  // T = J W with the clamped ray direction (Eq.2; reading C8)
  const double limx = 1.3 * (0.5 * c.width / (double)c.fx), limy = 1.3 * (0.5 * c.height / (double)c.fy);
  const double ux = fmin(limx, fmax(-limx, t[0] / tz)), uy = fmin(limy, fmax(-limy, t[1] / tz));
  const double J00 = c.fx / tz, J11 = c.fy / tz, J02 = -c.fx * ux / tz, J12 = -c.fy * uy / tz;
  double T[2][3], V[2][3];
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    T[0][b] = J00 * Wm[0][b] + J02 * Wm[2][b];
    T[1][b] = J11 * Wm[1][b] + J12 * Wm[2][b];
  }
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) V[a][b] = T[a][0] * Sg[0][b] + T[a][1] * Sg[1][b] + T[a][2] * Sg[2][b];  // T Sigma
  const double U00 = V[0][0] * T[0][0] + V[0][1] * T[0][1] + V[0][2] * T[0][2];
  const double U01 = V[0][0] * T[1][0] + V[0][1] * T[1][1] + V[0][2] * T[1][2];
  const double U11 = V[1][0] * T[1][0] + V[1][1] * T[1][1] + V[1][2] * T[1][2];
  // conic of the dilated covariance (Eq.3; reading C5; the Mip filter variant dilates by 0.1 instead of 0.3)
  const bool mip = VARIANT && (s.variant & GABSPLAT_VARIANT_MIP_FILTER) != 0;
  const bool line = VARIANT && (s.variant & GABSPLAT_VARIANT_LINE_INTEGRAL) != 0 && K > 0;
  const double dil = mip ? (double)kMipDilation : (double)kDilation;
  const double A = U00 + dil, C = U11 + dil;
  const double idet = 1.0 / (A * C - U01 * U01);
  const double ca = C * idet, cb = -U01 * idet, cc = A * idet;
  const float opac_in = s.opacities[i];
  reinterpret_cast<float4*>(out.conic_opacity)[i] = make_float4((float)ca, (float)cb, (float)cc, opac_in);
  // ---- variants (f4): both fold into the record the blend kernels gather, as an effective opacity o' and effective
  // weights u_k with  o' [(1 - sum u) + sum u cos] = o rho [(1 - sum w) + sum w C2 cos]:
  //   beta = 1 - sum_k w_k (1 - C2_k),  o' = o rho beta,  u_k = w_k C2_k / beta   (beta <= 0: M <= 0 everywhere, o' = 0)
  double o_eff = (double)opac_in;
  if (mip) o_eff *= sqrt(fmax(0.0, (U00 * U11 - U01 * U01) * idet));   // rho = sqrt(det U / det(U + 0.1 I))
  double att[VARIANT ? kMaxK : 1], beta = 1.0;
  if (VARIANT && line) {
    // C2_k = exp(-2 pi^2 (v.f_k)^2 / (v^T Sigma^-1 v)), v = W^T (u_x, u_y, 1) the world-space ray direction of J
    // (= f_z''^2 / S22 of Eq.25-27 for any completion of J's third row: DESIGN.md readings C2, C4)
    double v[3], b = 0.0;
#pragma unroll
    for (int m = 0; m < 3; ++m) v[m] = Wm[0][m] * ux + Wm[1][m] * uy + Wm[2][m];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const double rv = R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2];
      b += rv * rv / s2[j];
    }
    const double pi2 = 9.8696044010893586188;
    for (int k = 0; k < K; ++k) {
      const float* f = s.freqs + ((size_t)i * K + k) * 3;
      const double a = v[0] * (double)f[0] + v[1] * (double)f[1] + v[2] * (double)f[2];
      att[k] = exp(-2.0 * pi2 * a * a / b);
      beta -= (double)s.weights[(size_t)i * K + k] * (1.0 - att[k]);
    }
    o_eff = beta > 0.0 ? o_eff * beta : 0.0;
  }
  const float opac = (float)o_eff;
  // mu2D
  const double m2x = c.fx * t[0] / tz + c.cx, m2y = c.fy * t[1] / tz + c.cy;

  float* rec = out.packed + (size_t)i * packed_floats(K);
  reinterpret_cast<float4*>(rec)[0] =
      make_float4(m2.x, m2.y, (float)(m2x - (double)m2.x), (float)(m2y - (double)m2.y));
  {
    // conic = l l^T (Cholesky); q = -1/2 d^T conic d = -(u^2 + v^2) with L = l / sqrt(2)
    const double l11 = sqrt(ca), l21 = cb / l11, l22 = sqrt(fmax(cc - l21 * l21, 0.0));
    // ... and in base 2: G = 2^q with q = -(u^2 + v^2), L = l * sqrt(log2(e) / 2), so that the blend kernels feed q
    // straight to ex2 (no multiply by log2 e, no denormal guard: q >= qmin >= -8)
    const double rs = 0.84932180028801904272;  // sqrt(0.5 * log2(e))
    // envelope reject threshold: o G < 1/255  <=>  q < -ln(255 o); a little slack keeps the exact alpha test
    // the one that decides borderline pairs
    const float qmin = (float)((-log(255.0 * (double)opac) - 1e-4) * 1.4426950408889634074);  // in log2 units
    reinterpret_cast<float4*>(rec)[1] = make_float4((float)(l11 * rs), (float)(l21 * rs), (float)(l22 * rs), qmin);
  }
  // colour: max(0, 0.5 + sum_j Y_j(dir) sh_j), dir from the camera centre to the mean (reading C22)
  {
    double cp[3], v[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) cp[a] = -(Wm[0][a] * tau[0] + Wm[1][a] * tau[1] + Wm[2][a] * tau[2]);
#pragma unroll
    for (int a = 0; a < 3; ++a) v[a] = mu[a] - cp[a];
    const double il = 1.0 / sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    double Y[16];
    sh_values(s.sh_degree, v[0] * il, v[1] * il, v[2] * il, Y);
    const int nc = (s.sh_degree + 1) * (s.sh_degree + 1);
    double acc[3] = {0.5, 0.5, 0.5};
    const float4* shp = reinterpret_cast<const float4*>(s.sh + (size_t)i * 48);
    // 4 coefficients (12 floats) per 3 float4 loads
#pragma unroll
    for (int j4 = 0; j4 < 16; j4 += 4) {
      if (j4 >= nc) break;
      float buf[12];
#pragma unroll
      for (int v4 = 0; v4 < 3; ++v4) {
        const float4 x = shp[(j4 / 4) * 3 + v4];
        buf[4 * v4] = x.x; buf[4 * v4 + 1] = x.y; buf[4 * v4 + 2] = x.z; buf[4 * v4 + 3] = x.w;
      }
#pragma unroll
      for (int jj = 0; jj < 4; ++jj)
        if (j4 + jj < nc) {
#pragma unroll
          for (int ch = 0; ch < 3; ++ch) acc[ch] += Y[j4 + jj] * (double)buf[3 * jj + ch];
        }
    }
    uchar4 cl;
    cl.x = acc[0] < 0.0; cl.y = acc[1] < 0.0; cl.z = acc[2] < 0.0; cl.w = 0;
    const float r = cl.x ? 0.f : (float)acc[0], g = cl.y ? 0.f : (float)acc[1], b = cl.z ? 0.f : (float)acc[2];
    out.rgb[3 * i] = r; out.rgb[3 * i + 1] = g; out.rgb[3 * i + 2] = b;
    reinterpret_cast<uchar4*>(out.rgb_clamped)[i] = cl;
    reinterpret_cast<float4*>(rec)[2] = make_float4(opac, r, g, b);
  }
  // frequencies: f2D_k = U^-1 T Sigma f_k  (U undilated)
  {
    const double iu = 1.0 / (U00 * U11 - U01 * U01);
    const double two_pi = 6.283185307179586476925286766559;
    for (int k = 0; k < K; ++k) {
      const float* f = s.freqs + ((size_t)i * K + k) * 3;
      const double f0 = f[0], f1 = f[1], f2 = f[2];
      const double g0 = V[0][0] * f0 + V[0][1] * f1 + V[0][2] * f2;
      const double g1 = V[1][0] * f0 + V[1][1] * f1 + V[1][2] * f2;
      const double fx2 = (U11 * g0 - U01 * g1) * iu, fy2 = (U00 * g1 - U01 * g0) * iu;
      out.freq2d[((size_t)i * K + k) * 2] = (float)fx2;
      out.freq2d[((size_t)i * K + k) * 2 + 1] = (float)fy2;
      rec[12 + 2 * k] = (float)(two_pi * fx2);      // the blend kernels work in radians per pixel
      rec[12 + 2 * k + 1] = (float)(two_pi * fy2);
      const float wk = s.weights[(size_t)i * K + k];
      rec[12 + 2 * K + k] = (VARIANT && line) ? (beta > 0.0 ? (float)((double)wk * att[VARIANT ? k : 0] / beta) : 0.f) : wk;
    }
    for (int k = 3 * K; k < tail_floats(K); ++k) rec[12 + k] = 0.f;
  }
}

// Two kernels over chunks of kPreChunk consecutive primitives:
//  index_kernel  the fp32 indexing track of every primitive (coalesced loads; the depth test on the mean comes
//                first, so a primitive behind the camera costs 12 bytes): tiles_touched and radius for all, mean2d,
//                depth and rect for the visible ones, the number of visible primitives per chunk.  Few registers,
//                many warps per SM: it is a streaming kernel.
//  value_kernel  compacts the visible primitives of its chunk (from tiles_touched, in index order) and runs the fp64
//                value track over the compacted list.  In the paper-shaped scenes only 10-20 % of the primitives
//                are visible: without the compaction the value track runs with 3-6 live lanes per warp, and fused
//                with the indexing track its 128 registers hold the streaming part down to 16 warps per SM.
constexpr int kPreThreads = 256;
constexpr int kPreChunk = GABSPLAT_CHUNK;

__global__ void __launch_bounds__(kPreThreads) index_kernel(gabsplat_scene s, Camera c, gabsplat_projected out) {
  pdl_wait();
  __shared__ int s_n;
  __shared__ uint32_t s_kmin, s_kmax;
  if (threadIdx.x == 0) { s_n = 0; s_kmin = 0xffffffffu; s_kmax = 0u; }
  __syncthreads();
  const int base = blockIdx.x * kPreChunk;
  int mine = 0;
  uint32_t kmin = 0xffffffffu, kmax = 0u;  // bits(depth) of the visible primitives: what the binning sorts by
#pragma unroll 1
  for (int r = 0; r < kPreChunk / kPreThreads; ++r) {
    const int i = base + r * kPreThreads + threadIdx.x;
    if (i >= s.N) break;
    const float mx = s.means[3 * i], my = s.means[3 * i + 1], mz = s.means[3 * i + 2];
    const float tz = ffma(c.w[8], mx, ffma(c.w[9], my, ffma(c.w[10], mz, c.w[11])));
    uint32_t tiles = 0;
    int radius = 0;
    if (tz > c.z_near) {
      float sc[3], q[4];
#pragma unroll
      for (int a = 0; a < 3; ++a) sc[a] = s.scales[3 * i + a];
      const float4 qv = reinterpret_cast<const float4*>(s.rotations)[i];
      q[0] = qv.x; q[1] = qv.y; q[2] = qv.z; q[3] = qv.w;
      const Index ix = index_track(c, (s.variant & GABSPLAT_VARIANT_MIP_FILTER) ? kMipDilation : kDilation, mx, my, mz, sc, q);
      tiles = ix.tiles;
      radius = ix.radius;
      if (ix.visible) {
        ++mine;
        kmin = min(kmin, __float_as_uint(ix.depth));
        kmax = max(kmax, __float_as_uint(ix.depth));
        reinterpret_cast<float2*>(out.mean2d)[i] = make_float2(ix.m2x, ix.m2y);
        out.depth[i] = ix.depth;
        reinterpret_cast<int4*>(out.rect)[i] = make_int4(ix.x0, ix.y0, ix.x1, ix.y1);
      }
    }
    out.tiles_touched[i] = tiles;
    out.radius[i] = radius;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, d);
  kmin = __reduce_min_sync(0xffffffffu, kmin);
  kmax = __reduce_max_sync(0xffffffffu, kmax);
  if ((threadIdx.x & 31) == 0 && mine) { atomicAdd(&s_n, mine); atomicMin(&s_kmin, kmin); atomicMax(&s_kmax, kmax); }
  __syncthreads();
  if (threadIdx.x == 0) {
    out.chunk_visible[blockIdx.x] = (uint32_t)s_n;
    out.chunk_visible[gridDim.x + blockIdx.x] = s_kmin;
    out.chunk_visible[2 * gridDim.x + blockIdx.x] = s_kmax;
  }
}

constexpr int kValThreads = 128;

template <bool VARIANT>
__global__ void __launch_bounds__(kValThreads, 4) value_kernel(gabsplat_scene s, Camera c, gabsplat_projected out) {
  pdl_wait();
  __shared__ int s_i[kPreChunk];
  __shared__ int s_n;
  if (out.chunk_visible[blockIdx.x] == 0) return;
  if (threadIdx.x == 0) s_n = 0;
  __syncthreads();
  const int base = blockIdx.x * kPreChunk;
  for (int i = base + threadIdx.x; i < min(s.N, base + kPreChunk); i += kValThreads)
    if (out.tiles_touched[i] != 0) s_i[atomicAdd(&s_n, 1)] = i;
  __syncthreads();
  const int n = s_n;
  for (int j = threadIdx.x; j < n; j += kValThreads) value_track<VARIANT>(s, c, out, s_i[j]);
}

}  // namespace

// `value_stream` != st: the value track (needed only by the blend) runs there, so that the caller can overlap it
// with the binning, which needs only the indexing track; the caller orders the two streams with events.
cudaError_t launch_preprocess(const gabsplat_scene& s, const Camera& cam, const gabsplat_projected& out,
                              cudaStream_t st, cudaStream_t value_stream, cudaEvent_t index_done) {
  if (s.N == 0) return cudaSuccess;
  const int chunks = (s.N + kPreChunk - 1) / kPreChunk;
  launch_pdl(index_kernel, chunks, kPreThreads, 0, st, s, cam, out);
  if (value_stream != st) {
    cudaError_t e = cudaEventRecord(index_done, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(value_stream, index_done, 0);
    if (e != cudaSuccess) return e;
  }
  if (s.variant) launch_pdl(value_kernel<true>, chunks, kValThreads, 0, value_stream, s, cam, out);
  else launch_pdl(value_kernel<false>, chunks, kValThreads, 0, value_stream, s, cam, out);
  launched(2);
  return cudaGetLastError();
}

}  // namespace gabsplat
