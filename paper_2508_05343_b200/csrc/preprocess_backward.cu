// S4b / K8: chain rule from the projected quantities back to the primitive parameters (the paper gives no
// equations -- PAPER.md:48, :129; derivation in DESIGN.md "Backward", per-primitive part):
//   conic -> U;  f2D = U^-1 T Sigma f -> (U, T, Sigma, f);  U = T Sigma T^T -> (T, Sigma);  T = J W -> J -> t;
//   mu2D -> t;  t -> mu;  Sigma = R S S^T R^T -> (scale, quaternion);  rgb -> (SH, mu through the view direction).
// Evaluated in fp64 (HBM-bound: the arithmetic is free, see preprocess.cu).  The kernel zeroes the gradient
// arrays are zeroed by a separate store-only kernel that overlaps the blend backward on a side stream.
#include "common.cuh"
#include "sh.cuh"

namespace gabsplat {
namespace {

// chain rule of one visible primitive (fp64); writes its row of every gradient array
template <bool VARIANT>
__device__ __forceinline__ void backward_one(const gabsplat_scene& s, const Camera& c, const uint8_t* __restrict__ rgb_clamped,
                                             float* grad2d, const gabsplat_grads& g, const int i) {
  const int K = s.K;
  const int G = grad2d_floats(K);
  const float* g2 = grad2d + (size_t)i * G;

  double Wm[3][3], tau[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
#pragma unroll
    for (int b = 0; b < 3; ++b) Wm[a][b] = (double)c.w[4 * a + b];
    tau[a] = (double)c.w[4 * a + 3];
  }
  const double mu[3] = {(double)s.means[3 * i], (double)s.means[3 * i + 1], (double)s.means[3 * i + 2]};
  double t[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) t[a] = Wm[a][0] * mu[0] + Wm[a][1] * mu[1] + Wm[a][2] * mu[2] + tau[a];
  const double tz = t[2];
  const double sc[3] = {(double)s.scales[3 * i], (double)s.scales[3 * i + 1], (double)s.scales[3 * i + 2]};
  const double qw = s.rotations[4 * i], qx = s.rotations[4 * i + 1], qy = s.rotations[4 * i + 2], qz = s.rotations[4 * i + 3];
  const double R[3][3] = {{1 - 2 * (qy * qy + qz * qz), 2 * (qx * qy - qw * qz), 2 * (qx * qz + qw * qy)},
                          {2 * (qx * qy + qw * qz), 1 - 2 * (qx * qx + qz * qz), 2 * (qy * qz - qw * qx)},
                          {2 * (qx * qz - qw * qy), 2 * (qy * qz + qw * qx), 1 - 2 * (qx * qx + qy * qy)}};
  double Sg[3][3];
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b)
      Sg[a][b] = R[a][0] * sc[0] * sc[0] * R[b][0] + R[a][1] * sc[1] * sc[1] * R[b][1] + R[a][2] * sc[2] * sc[2] * R[b][2];
  const double limx = 1.3 * (0.5 * c.width / (double)c.fx), limy = 1.3 * (0.5 * c.height / (double)c.fy);
  const double rx = t[0] / tz, ry = t[1] / tz;
  const bool clampx = rx < -limx || rx > limx, clampy = ry < -limy || ry > limy;
  const double ux = fmin(limx, fmax(-limx, rx)), uy = fmin(limy, fmax(-limy, ry));
  const double fx = c.fx, fy = c.fy;
  const double J00 = fx / tz, J11 = fy / tz, J02 = -fx * ux / tz, J12 = -fy * uy / tz;
  double T[2][3], V[2][3];
#pragma unroll
  for (int b = 0; b < 3; ++b) {
    T[0][b] = J00 * Wm[0][b] + J02 * Wm[2][b];
    T[1][b] = J11 * Wm[1][b] + J12 * Wm[2][b];
  }
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 3; ++b) V[a][b] = T[a][0] * Sg[0][b] + T[a][1] * Sg[1][b] + T[a][2] * Sg[2][b];
  const double U00 = V[0][0] * T[0][0] + V[0][1] * T[0][1] + V[0][2] * T[0][2];
  const double U01 = V[0][0] * T[1][0] + V[0][1] * T[1][1] + V[0][2] * T[1][2];
  const double U11 = V[1][0] * T[1][0] + V[1][1] * T[1][1] + V[1][2] * T[1][2];
  const bool mip = VARIANT && (s.variant & GABSPLAT_VARIANT_MIP_FILTER) != 0;
  const bool line = VARIANT && (s.variant & GABSPLAT_VARIANT_LINE_INTEGRAL) != 0 && K > 0;
  const double dil = mip ? (double)kMipDilation : (double)kDilation;
  const double A = U00 + dil, C = U11 + dil;
  const double idet = 1.0 / (A * C - U01 * U01);
  const double ca = C * idet, cb = -U01 * idet, cc = A * idet;
  // ---- variants (f4; preprocess.cu value_track): the blend saw o' = o rho beta and u_k = w_k C2_k / beta
  const double opac = (double)s.opacities[i];
  const double rho = mip ? sqrt(fmax(0.0, (U00 * U11 - U01 * U01) * idet)) : 1.0;
  constexpr int KV = VARIANT ? kMaxK : 1;
  double att[KV], av[KV], beta = 1.0, v[3] = {0, 0, 0}, yv[3] = {0, 0, 0}, bq = 1.0;
#pragma unroll
  for (int k = 0; k < KV; ++k) { att[k] = 1.0; av[k] = 0.0; }
  if (VARIANT && line) {
#pragma unroll
    for (int m = 0; m < 3; ++m) v[m] = Wm[0][m] * ux + Wm[1][m] * uy + Wm[2][m];
    // y = Sigma^-1 v = R diag(1/s^2) R^T v,  b = v^T y
    double rv[3];
    bq = 0.0;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      rv[j] = (R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2]) / (sc[j] * sc[j]);
      bq += rv[j] * (R[0][j] * v[0] + R[1][j] * v[1] + R[2][j] * v[2]);
    }
#pragma unroll
    for (int m = 0; m < 3; ++m) yv[m] = R[m][0] * rv[0] + R[m][1] * rv[1] + R[m][2] * rv[2];
    const double pi2 = 9.8696044010893586188;
    for (int k = 0; k < K; ++k) {
      const float* fp = s.freqs + ((size_t)i * K + k) * 3;
      av[k] = v[0] * (double)fp[0] + v[1] * (double)fp[1] + v[2] * (double)fp[2];
      att[k] = exp(-2.0 * pi2 * av[k] * av[k] / bq);
      beta -= (double)s.weights[(size_t)i * K + k] * (1.0 - att[k]);
    }
  }
  const bool live = !line || beta > 0.0;   // beta <= 0: the primitive was never blended, its 2D record is zero
  const double g_oeff = live ? (double)g2[5] : 0.0;
  // d o' -> (o, rho, beta);  d u_k -> (w_k, C2_k, beta)
  double g_beta = g_oeff * opac * rho, g_att[KV];
#pragma unroll
  for (int k = 0; k < KV; ++k) g_att[k] = 0.0;
  double g_w[KV];
  for (int k = 0; VARIANT && k < K; ++k) {
    const double gu = live ? (double)g2[9 + 2 * K + k] : 0.0;
    if (line) {
      const double w = (double)s.weights[(size_t)i * K + k];
      const double ib = live ? 1.0 / beta : 0.0;
      g_beta -= gu * (w * att[k] * ib) * ib;
      g_w[k] = gu * att[k] * ib;
      g_att[k] = gu * w * ib;
    } else {
      g_w[k] = gu;
    }
  }
  if (VARIANT && line) {
    for (int k = 0; k < K; ++k) {
      const double w = (double)s.weights[(size_t)i * K + k];
      g_w[k] -= g_beta * (1.0 - att[k]);
      g_att[k] += g_beta * w;
    }
  }
  const double g_opacity = g_oeff * rho * (line ? beta : 1.0);
  const double g_rho = g_oeff * opac * (line ? beta : 1.0);

  // conic -> U_d (= U + const).  The blend accumulated S = sum gq w w^T with w = L^T d the whitened pixel offset
  // (L = sqrt(log2(e) / 2) * Cholesky factor of the conic, as packed for the blend) and gq = dL/d(ln G).  With
  // G_c = sum gq (-1/2 d d^T):  G_U = -C G_c C = 1/2 sum gq (C d)(C d)^T = 2 ln^2(2) L S L^T.
  double GU[2][2];
  {
    const double rs = 0.84932180028801904272;  // sqrt(0.5 * log2(e)), as in preprocess.cu
    const double l11 = sqrt(ca), l21 = cb / l11, l22 = sqrt(fmax(cc - l21 * l21, 0.0));
    const double L11 = l11 * rs, L21 = l21 * rs, L22 = l22 * rs;
    const double suu = g2[2], suv = g2[3], svv = g2[4];
    // M = L S  (L = [[L11, 0], [L21, L22]])
    const double m00 = L11 * suu, m01 = L11 * suv;
    const double m10 = L21 * suu + L22 * suv, m11 = L21 * suv + L22 * svv;
    const double k = 2.0 * 0.69314718055994530942 * 0.69314718055994530942;
    GU[0][0] = k * (m00 * L11);
    GU[0][1] = k * (m00 * L21 + m01 * L22);
    GU[1][0] = k * (m10 * L11);
    GU[1][1] = k * (m10 * L21 + m11 * L22);
  }
  double gS[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, gT[2][3] = {{0, 0, 0}, {0, 0, 0}};
  double gt[3] = {0, 0, 0};
  double gf_extra[KV][3];
#pragma unroll
  for (int k = 0; k < KV; ++k) gf_extra[k][0] = gf_extra[k][1] = gf_extra[k][2] = 0.0;
  // a primitive outside the value contract (a scale of exactly 0) has b = inf: C2_k = 1 whatever f and v are, no gradient
  // flows through it -- and 0 * inf below would turn the whole row into NaN
  if (VARIANT && line && live && bq > 0.0 && bq < 1e300) {
    // C2_k = exp(-2 pi^2 a_k^2 / b), a_k = v . f_k, b = v^T Sigma^-1 v, v = W^T (u_x, u_y, 1)
    const double pi2 = 9.8696044010893586188;
    double gv[3] = {0, 0, 0}, gb = 0.0;
    for (int k = 0; k < K; ++k) {
      const float* fp = s.freqs + ((size_t)i * K + k) * 3;
      const double gl = g_att[k] * att[k];  // dL/d(ln C2_k)
      const double ga = gl * (-4.0 * pi2 * av[k] / bq);
      gb += gl * (2.0 * pi2 * av[k] * av[k] / (bq * bq));
#pragma unroll
      for (int m = 0; m < 3; ++m) { gf_extra[k][m] = ga * v[m]; gv[m] += ga * (double)fp[m]; }
    }
#pragma unroll
    for (int m = 0; m < 3; ++m) gv[m] += 2.0 * gb * yv[m];
#pragma unroll
    for (int m = 0; m < 3; ++m)
#pragma unroll
      for (int n = 0; n < 3; ++n) gS[m][n] -= gb * yv[m] * yv[n];  // d(Sigma^-1) = -Sigma^-1 dSigma Sigma^-1
    const double gcx = Wm[0][0] * gv[0] + Wm[0][1] * gv[1] + Wm[0][2] * gv[2];
    const double gcy = Wm[1][0] * gv[0] + Wm[1][1] * gv[1] + Wm[1][2] * gv[2];
    if (!clampx) { gt[0] += gcx / tz; gt[2] -= gcx * t[0] / (tz * tz); }
    if (!clampy) { gt[1] += gcy / tz; gt[2] -= gcy * t[1] / (tz * tz); }
  }
  // f2D_k = U^-1 T Sigma f_k  (U undilated)
  {
    const double iu = 1.0 / (U00 * U11 - U01 * U01);
    const double Ui00 = U11 * iu, Ui01 = -U01 * iu, Ui11 = U00 * iu;
    if (mip && rho > 0.0) {  // rho = sqrt(det U / det U_d):  d rho = rho / 2 tr((U^-1 - U_d^-1) dU); rho = 0 (det U = 0,
                             // a degenerate primitive): never blended, and U^-1 is not finite
      const double h = 0.5 * g_rho * rho;
      GU[0][0] += h * (Ui00 - ca); GU[0][1] += h * (Ui01 - cb); GU[1][0] += h * (Ui01 - cb); GU[1][1] += h * (Ui11 - cc);
    }
    const double two_pi = 6.283185307179586476925286766559;  // grad2d holds d/d(2 pi f2D)
    for (int k = 0; k < K; ++k) {
      const float* fp = s.freqs + ((size_t)i * K + k) * 3;
      const double f[3] = {fp[0], fp[1], fp[2]};
      const double gf0 = two_pi * (double)g2[9 + 2 * k], gf1 = two_pi * (double)g2[9 + 2 * k + 1];
      const double h0 = Ui00 * gf0 + Ui01 * gf1, h1 = Ui01 * gf0 + Ui11 * gf1;
      const double b0 = V[0][0] * f[0] + V[0][1] * f[1] + V[0][2] * f[2];
      const double b1 = V[1][0] * f[0] + V[1][1] * f[1] + V[1][2] * f[2];
      const double f2x = Ui00 * b0 + Ui01 * b1, f2y = Ui01 * b0 + Ui11 * b1;
      GU[0][0] -= h0 * f2x;
      GU[0][1] -= 0.5 * (h0 * f2y + f2x * h1);
      GU[1][0] -= 0.5 * (h1 * f2x + f2y * h0);
      GU[1][1] -= h1 * f2y;
      double Th[3], Sf[3];
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        Th[m] = T[0][m] * h0 + T[1][m] * h1;
        Sf[m] = Sg[m][0] * f[0] + Sg[m][1] * f[1] + Sg[m][2] * f[2];
      }
#pragma unroll
      for (int m = 0; m < 3; ++m)
#pragma unroll
        for (int n = 0; n < 3; ++n) gS[m][n] += 0.5 * (Th[m] * f[n] + f[m] * Th[n]);
#pragma unroll
      for (int m = 0; m < 3; ++m) { gT[0][m] += h0 * Sf[m]; gT[1][m] += h1 * Sf[m]; }
#pragma unroll
      for (int m = 0; m < 3; ++m)
        g.d_freqs[((size_t)i * K + k) * 3 + m] = (float)(Sg[m][0] * Th[0] + Sg[m][1] * Th[1] + Sg[m][2] * Th[2] + (VARIANT ? gf_extra[VARIANT ? k : 0][m] : 0.0));
      g.d_weights[(size_t)i * K + k] = VARIANT ? (float)g_w[VARIANT ? k : 0] : g2[9 + 2 * K + k];
    }
  }
  // U = T Sigma T^T
  {
    double GUT[2][3];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int m = 0; m < 3; ++m) GUT[r][m] = GU[r][0] * T[0][m] + GU[r][1] * T[1][m];
#pragma unroll
    for (int m = 0; m < 3; ++m)
#pragma unroll
      for (int n = 0; n < 3; ++n) gS[m][n] += T[0][m] * GUT[0][n] + T[1][m] * GUT[1][n];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int m = 0; m < 3; ++m) gT[r][m] += 2.0 * (GUT[r][0] * Sg[0][m] + GUT[r][1] * Sg[1][m] + GUT[r][2] * Sg[2][m]);
  }
  // T = J W  ->  g_J = g_T W^T;  J(t) and mu2D(t)
  {
    double gJ[2][3];
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int m = 0; m < 3; ++m) gJ[r][m] = gT[r][0] * Wm[m][0] + gT[r][1] * Wm[m][1] + gT[r][2] * Wm[m][2];
    const double iz = 1.0 / tz, iz2 = iz * iz;
    gt[2] += -gJ[0][0] * fx * iz2 - gJ[1][1] * fy * iz2;
    gt[2] += gJ[0][2] * fx * ux * iz2 + gJ[1][2] * fy * uy * iz2;
    if (!clampx) { gt[0] += -gJ[0][2] * fx * iz2; gt[2] += gJ[0][2] * fx * t[0] * iz2 * iz; }
    if (!clampy) { gt[1] += -gJ[1][2] * fy * iz2; gt[2] += gJ[1][2] * fy * t[1] * iz2 * iz; }
    const double gmx = g2[0], gmy = g2[1];
    gt[0] += gmx * fx * iz;
    gt[1] += gmy * fy * iz;
    gt[2] += -(gmx * fx * t[0] + gmy * fy * t[1]) * iz2;
  }
  double gmu[3];
#pragma unroll
  for (int m = 0; m < 3; ++m) gmu[m] = Wm[0][m] * gt[0] + Wm[1][m] * gt[1] + Wm[2][m] * gt[2];
  // Sigma = Ms Ms^T, Ms = R diag(s):  g_Ms = 2 g_Sigma Ms
  {
    double gR[3][3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
      double gs = 0.0;
#pragma unroll
      for (int m = 0; m < 3; ++m) {
        const double gMs = 2.0 * (gS[m][0] * R[0][n] + gS[m][1] * R[1][n] + gS[m][2] * R[2][n]) * sc[n];
        gs += R[m][n] * gMs;
        gR[m][n] = gMs * sc[n];
      }
      g.d_scales[3 * i + n] = (float)gs;
    }
    // R(q) polynomial (un-normalised) form
    const double dw = 2 * (-qz * gR[0][1] + qy * gR[0][2] + qz * gR[1][0] - qx * gR[1][2] - qy * gR[2][0] + qx * gR[2][1]);
    const double dx = 2 * (qy * gR[0][1] + qz * gR[0][2] + qy * gR[1][0] - 2 * qx * gR[1][1] - qw * gR[1][2] + qz * gR[2][0] +
                           qw * gR[2][1] - 2 * qx * gR[2][2]);
    const double dy = 2 * (-2 * qy * gR[0][0] + qx * gR[0][1] + qw * gR[0][2] + qx * gR[1][0] + qz * gR[1][2] - qw * gR[2][0] +
                           qz * gR[2][1] - 2 * qy * gR[2][2]);
    const double dz = 2 * (-2 * qz * gR[0][0] - qw * gR[0][1] + qx * gR[0][2] + qw * gR[1][0] - 2 * qz * gR[1][1] + qy * gR[1][2] +
                           qx * gR[2][0] + qy * gR[2][1]);
    reinterpret_cast<float4*>(g.d_rotations)[i] = make_float4((float)dw, (float)dx, (float)dy, (float)dz);
  }
  // colour: rgb = max(0, 0.5 + sum_j Y_j(dir) sh_j)
  {
    double cp[3], v[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) cp[a] = -(Wm[0][a] * tau[0] + Wm[1][a] * tau[1] + Wm[2][a] * tau[2]);
#pragma unroll
    for (int a = 0; a < 3; ++a) v[a] = mu[a] - cp[a];
    const double il = 1.0 / sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    const double d[3] = {v[0] * il, v[1] * il, v[2] * il};
    double Y[16], dY[16][3];
    sh_values(s.sh_degree, d[0], d[1], d[2], Y);
    sh_gradients(s.sh_degree, d[0], d[1], d[2], dY);
    const int nc = (s.sh_degree + 1) * (s.sh_degree + 1);
    const uchar4 cl = reinterpret_cast<const uchar4*>(rgb_clamped)[i];
    const double gr[3] = {cl.x ? 0.0 : (double)g2[6], cl.y ? 0.0 : (double)g2[7], cl.z ? 0.0 : (double)g2[8]};
    double gd[3] = {0, 0, 0};
    const float4* shp = reinterpret_cast<const float4*>(s.sh + (size_t)i * 48);
    float4* dsh = reinterpret_cast<float4*>(g.d_sh + (size_t)i * 48);
    // 4 coefficients (12 floats) per 3 vector loads / stores; rows >= nc stay zero
#pragma unroll
    for (int j4 = 0; j4 < 16; j4 += 4) {
      if (j4 >= nc) break;
      float in[12], o[12];
#pragma unroll
      for (int v4 = 0; v4 < 3; ++v4) {
        const float4 x = shp[(j4 / 4) * 3 + v4];
        in[4 * v4] = x.x; in[4 * v4 + 1] = x.y; in[4 * v4 + 2] = x.z; in[4 * v4 + 3] = x.w;
      }
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) {
        const bool live = j4 + jj < nc;
        double dot = 0.0;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
          o[3 * jj + ch] = live ? (float)(Y[j4 + jj] * gr[ch]) : 0.f;
          dot += (double)in[3 * jj + ch] * gr[ch];
        }
        if (live) {
#pragma unroll
          for (int m = 0; m < 3; ++m) gd[m] += dY[j4 + jj][m] * dot;
        }
      }
#pragma unroll
      for (int v4 = 0; v4 < 3; ++v4) dsh[(j4 / 4) * 3 + v4] = make_float4(o[4 * v4], o[4 * v4 + 1], o[4 * v4 + 2], o[4 * v4 + 3]);
    }
    const double dg = d[0] * gd[0] + d[1] * gd[1] + d[2] * gd[2];
#pragma unroll
    for (int m = 0; m < 3; ++m) gmu[m] += (gd[m] - d[m] * dg) * il;
  }
#pragma unroll
  for (int m = 0; m < 3; ++m) g.d_means[3 * i + m] = (float)gmu[m];
  g.d_opacities[i] = (float)g_opacity;
  if (g.d_mean2d) { g.d_mean2d[2 * i] = g2[0]; g.d_mean2d[2 * i + 1] = g2[1]; }
  if (g.d_mean2d_abs) { g.d_mean2d_abs[2 * i] = g2[9 + 3 * K]; g.d_mean2d_abs[2 * i + 1] = g2[10 + 3 * K]; }
  // clear the primitive's 2D gradient record: the workspace is all zero again when the call returns (only visible
  // primitives ever have a non-zero record), so no 96 B x N memset is needed before the next blend backward
  float4* row = reinterpret_cast<float4*>(grad2d + (size_t)i * G);
  for (int q = 0; q < G / 4; ++q) row[q] = make_float4(0.f, 0.f, 0.f, 0.f);
}

constexpr int kBwdThreads = 128;

// One thread per VISIBLE primitive: rank r of the binning's depth-ordered list (any order would do; the list is
// there, compact, and keeps every lane of every live warp busy -- 10-20 % of the primitives are visible).  The
// gradient arrays were zeroed by grad_zero_kernel (side stream, concurrently with the blend backward); rows of
// culled primitives stay zero.
#ifndef GS_PBWD_MINB
#define GS_PBWD_MINB 3
#endif
template <bool VARIANT>
__global__ void __launch_bounds__(kBwdThreads, GS_PBWD_MINB) preprocess_backward_kernel(gabsplat_scene s, Camera c, const uint32_t* __restrict__ order,
                                                                         const uint32_t* __restrict__ n_vis,
                                                                         const uint8_t* __restrict__ rgb_clamped,
                                                                         float* grad2d, gabsplat_grads g) {
  pdl_wait();
  const uint32_t r = blockIdx.x * kBwdThreads + threadIdx.x;
  if (r >= *n_vis) return;
  backward_one<VARIANT>(s, c, rgb_clamped, grad2d, g, (int)order[r]);
}

// Zeroes every gradient array (coalesced 16-byte stores, grid-stride): 300 B per primitive of pure HBM writes,
// launched on a side stream so that it overlaps the ALU-bound blend backward.
__global__ void __launch_bounds__(256) grad_zero_kernel(int N, int K, gabsplat_grads g) {
  const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
  auto fill = [&](float* p, size_t n) {  // p is 16-byte aligned; n floats
    if (!p) return;
    float4* p4 = reinterpret_cast<float4*>(p);
    const size_t n4 = n / 4, stride = (size_t)gridDim.x * blockDim.x, t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (size_t j = t; j < n4; j += stride) p4[j] = z;
    for (size_t j = 4 * n4 + t; j < n; j += stride) p[j] = 0.f;
  };
  const size_t n = (size_t)N, k = (size_t)K;
  fill(g.d_sh, 48 * n);
  fill(g.d_means, 3 * n);
  fill(g.d_scales, 3 * n);
  fill(g.d_rotations, 4 * n);
  fill(g.d_opacities, n);
  if (K) { fill(g.d_freqs, 3 * k * n); fill(g.d_weights, k * n); }
  fill(g.d_mean2d, 2 * n);
  fill(g.d_mean2d_abs, 2 * n);
}

}  // namespace

cudaError_t launch_grad_zero(const gabsplat_scene& s, const gabsplat_grads& g, cudaStream_t st) {
  if (s.N == 0) return cudaSuccess;
  grad_zero_kernel<<<sm_count() * 8, 256, 0, st>>>(s.N, s.K, g);
  launched();
  return cudaGetLastError();
}

cudaError_t launch_preprocess_backward(const gabsplat_scene& s, const Camera& cam, const gabsplat_projected& proj,
                                       const gabsplat_binning& bin, float* grad2d, const gabsplat_grads& g, cudaStream_t st) {
  if (s.N == 0) return cudaGetLastError();
  const uint32_t *order, *n_vis;
  binning_visible_list(bin, s.N, cam.tiles_x * cam.tiles_y, &order, &n_vis);
  if (s.variant)
    launch_pdl(preprocess_backward_kernel<true>, (s.N + kBwdThreads - 1) / kBwdThreads, kBwdThreads, 0, st, s, cam, order, n_vis,
               (const uint8_t*)proj.rgb_clamped, grad2d, g);
  else
    launch_pdl(preprocess_backward_kernel<false>, (s.N + kBwdThreads - 1) / kBwdThreads, kBwdThreads, 0, st, s, cam, order, n_vis,
               (const uint8_t*)proj.rgb_clamped, grad2d, g);
  launched();
  return cudaGetLastError();
}

}  // namespace gabsplat
