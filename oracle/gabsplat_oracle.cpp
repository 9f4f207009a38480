// ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// A plain, slow, double-precision CPU renderer for 3D Gabor-based primitives (3DGabSplat,
// arXiv 2508.05343), written from the paper's equations; forward image and analytic gradients.
// It shares no code, header, table or constant generator with the CUDA path under
// paper_2508_05343_b200/csrc/.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.
//
// What it computes (citations are /root/reference/PAPER.md line + equation):
//   * primitive:   Gabor_k(x) = G_k(x) [ (1 - sum_i w_i) + sum_i w_i cos(2 pi f_i^T (x - mu)) ]   :127 Eq.7
//   * projection:  Sigma' = J W Sigma W^T J^T, top-left 2x2 kept                                   :91 Eq.2, :93-99
//   * frequency:   f_proj^T = f^T (JW)^-1  (supplementary form, reading C1)          :145 Eq.9, :414
//                  f2D = (f_proj_x - S02/S22 f_proj_z, f_proj_y - S12/S22 f_proj_z), S = Sigma''^-1  :150-154 Eq.10-11, :496 Eq.29
//   * 2D primitive: G2D(x) [ (1 - sum w) + sum w cos(2 pi f2D . (x - mu2D)) ]                      :158 Eq.12
//   * blending:    C(x) = sum_i c_i a_i prod_{j<i} (1 - a_j),  a_i = o_i Gabor2D_i(x), depth order  :162 Eq.13, :103
// Everything the paper leaves to "the tile-based rasterizer from 3DGS" (:160) -- dilation, the
// 1/255 and 0.99 alpha rules, the 1e-4 transmittance stop, 3-sigma tile rectangles, SH colour --
// follows the readings C5-C23 listed in DESIGN.md.
//
// Precision: all VALUES are double.  INTEGER decisions that the CUDA path must reproduce bit for
// bit (visibility, depth key, radius, tile rectangle) are taken in float32 by the "indexing twin"
// below, a normative float32 operation sequence; this file
// is compiled with -ffp-contract=off so every fused multiply-add is an explicit std::fmaf.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): single on-axis isotropic primitive closed form;
// two-primitive Eq.13 written out; w=0 / f=0 equals an independently written numpy Gaussian
// compositor (:131); phase invariance of Eq.16-17 off axis; f2D independent of J's third row;
// z-quadrature of the ray-space 3D Gabor (:420-497); partition of unity; permutation and
// component-split invariance; SH Gram matrix by quadrature; brute-force tile lists;
// central finite differences for all seven gradient groups.
//
// Parity unpinned: full-size images have no external pin beyond the above.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <omp.h>

namespace {

constexpr int KMAX = 8;
constexpr int TILE = 16;
constexpr double DILATION = 0.3;          // reading C5
constexpr double ALPHA_MAX = 0.99;        // reading C8
constexpr double ALPHA_MIN = 1.0 / 255.0; // reading C8
constexpr double T_MIN = 1e-4;            // reading C8
constexpr double TWO_PI = 6.283185307179586476925286766559;

// Variants of the primitive, bit flags:
//  VARIANT_LINE_INTEGRAL  keep the per-component amplitude of the exact line integral along the ray that Eq.12 drops
//      (Eq.25-27): component k is attenuated by C2_k = exp(-2 pi^2 (f_z'')^2 / S22), f_z'' the z
//      component of f_proj (Eq.9) and S22 the zz entry of the inverse ray-space covariance (Eq.19).  The constants
//      printed at :483 are garbled (C2 is printed with a positive exponent, C1 as a reciprocal); completing the
//      square in Eq.24 gives the value used here (reading C4; pinned by the z-quadrature test).  The
//      common factor C1 is dropped as in Eq.12, so the Gaussian term keeps weight 1 - sum w and a primitive with
//      f = 0 is unchanged:  M = (1 - sum_k w_k) + sum_k w_k C2_k cos(phi_k).
//  VARIANT_MIP_FILTER     the 2D Mip filter of Mip-Splatting in place of the 0.3 px^2 dilation (the
//      "+Mip-Splatting+AbsGS" variant): the 2D covariance is dilated by 0.1 px^2 and the opacity is scaled by
//      sqrt(det U / det(U + 0.1 I)) so that the splat keeps its integral.
constexpr int VARIANT_LINE_INTEGRAL = 1, VARIANT_MIP_FILTER = 2;
constexpr double MIP_DILATION = 0.1;

struct Scene {
    int N, K, deg;
    const float *means, *scales, *quats, *opac, *sh, *freqs, *weights;
    int variant = 0;
};

struct Cam {
    int W, H;
    double fx, fy, cx, cy;
    double Wm[3][3], tau[3];
    double z_near, bg[3];
    int gx, gy;
};

Cam load_cam(const double* c) {
    Cam k;
    k.W = (int)c[0]; k.H = (int)c[1];
    k.fx = c[2]; k.fy = c[3]; k.cx = c[4]; k.cy = c[5];
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) k.Wm[i][j] = c[6 + 4 * i + j];
        k.tau[i] = c[6 + 4 * i + 3];
    }
    k.z_near = c[18];
    k.bg[0] = c[19]; k.bg[1] = c[20]; k.bg[2] = c[21];
    k.gx = (k.W + TILE - 1) / TILE;
    k.gy = (k.H + TILE - 1) / TILE;
    return k;
}

// ---------------------------------------------------------------------------------------------
// Indexing twin: float32, normative operation order.  Decides visibility, depth key,
// radius and tile rectangle.  Every line is one IEEE-754 correctly rounded operation (or fmaf).
// ---------------------------------------------------------------------------------------------
struct Twin {
    bool visible;
    uint32_t depth_bits;
    float mean2d[2];
    int radius;
    int rect[4];  // xmin, ymin, xmax (exclusive), ymax (exclusive), in tiles
    uint32_t tiles;
};

inline float clampf(float v, float lo, float hi) { return std::fmin(std::fmax(v, lo), hi); }

Twin twin_index(const Scene& s, const Cam& c, int i) {
    Twin o{};
    float Wf[3][3], tf[3];
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) Wf[a][b] = (float)c.Wm[a][b];
    const float mx = s.means[3 * i], my = s.means[3 * i + 1], mz = s.means[3 * i + 2];
    for (int a = 0; a < 3; ++a)
        tf[a] = std::fmaf(Wf[a][0], mx, std::fmaf(Wf[a][1], my, std::fmaf(Wf[a][2], mz, (float)c.tau[a])));
    if (!(tf[2] > (float)c.z_near)) return o;

    // R(q), M = R diag(s), Sigma = M M^T
    const float qw = s.quats[4 * i], qx = s.quats[4 * i + 1], qy = s.quats[4 * i + 2], qz = s.quats[4 * i + 3];
    float R[3][3];
    R[0][0] = 1.0f - 2.0f * (qy * qy + qz * qz);
    R[0][1] = 2.0f * (qx * qy - qw * qz);
    R[0][2] = 2.0f * (qx * qz + qw * qy);
    R[1][0] = 2.0f * (qx * qy + qw * qz);
    R[1][1] = 1.0f - 2.0f * (qx * qx + qz * qz);
    R[1][2] = 2.0f * (qy * qz - qw * qx);
    R[2][0] = 2.0f * (qx * qz - qw * qy);
    R[2][1] = 2.0f * (qy * qz + qw * qx);
    R[2][2] = 1.0f - 2.0f * (qx * qx + qy * qy);
    float M[3][3], Sg[3][3];
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) M[a][b] = R[a][b] * s.scales[3 * i + b];
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
        Sg[a][b] = std::fmaf(M[a][2], M[b][2], std::fmaf(M[a][1], M[b][1], M[a][0] * M[b][0]));

    // J (2x3) with the clamped ray direction, T = J W
    const float fx = (float)c.fx, fy = (float)c.fy;
    const float limx = 1.3f * ((0.5f * (float)c.W) / fx), limy = 1.3f * ((0.5f * (float)c.H) / fy);
    const float ux = clampf(tf[0] / tf[2], -limx, limx), uy = clampf(tf[1] / tf[2], -limy, limy);
    const float J00 = fx / tf[2], J11 = fy / tf[2];
    const float J02 = -(J00 * ux), J12 = -(J11 * uy);
    float T[2][3], V[2][3];
    for (int b = 0; b < 3; ++b) {
        T[0][b] = std::fmaf(J02, Wf[2][b], J00 * Wf[0][b]);
        T[1][b] = std::fmaf(J12, Wf[2][b], J11 * Wf[1][b]);
    }
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 3; ++b)
        V[a][b] = std::fmaf(T[a][2], Sg[2][b], std::fmaf(T[a][1], Sg[1][b], T[a][0] * Sg[0][b]));
    const float U00 = std::fmaf(V[0][2], T[0][2], std::fmaf(V[0][1], T[0][1], V[0][0] * T[0][0]));
    const float U01 = std::fmaf(V[0][2], T[1][2], std::fmaf(V[0][1], T[1][1], V[0][0] * T[1][0]));
    const float U11 = std::fmaf(V[1][2], T[1][2], std::fmaf(V[1][1], T[1][1], V[1][0] * T[1][0]));
    const float dil = (s.variant & VARIANT_MIP_FILTER) ? 0.1f : 0.3f;
    const float A = U00 + dil, C = U11 + dil;
    const float det = A * C - U01 * U01;
    if (!(det > 0.0f)) return o;
    // lambda_max = mid + sqrt(((A-C)/2)^2 + B^2)   (reading C9); radius = ceil(3 sqrt(lambda_max))
    const float mid = 0.5f * (A + C), hd = 0.5f * (A - C);
    const float lam = mid + std::sqrt(std::fmaf(hd, hd, U01 * U01));
    const float rf = std::ceil(3.0f * std::sqrt(lam));
    const float m2x = std::fmaf(fx, tf[0] / tf[2], (float)c.cx), m2y = std::fmaf(fy, tf[1] / tf[2], (float)c.cy);
    // tile rectangle (reading C10)
    const float gxf = (float)c.gx, gyf = (float)c.gy;
    o.rect[0] = (int)clampf((m2x - rf) * 0.0625f, 0.0f, gxf);
    o.rect[1] = (int)clampf((m2y - rf) * 0.0625f, 0.0f, gyf);
    o.rect[2] = (int)clampf(((m2x + rf) + 15.0f) * 0.0625f, 0.0f, gxf);
    o.rect[3] = (int)clampf(((m2y + rf) + 15.0f) * 0.0625f, 0.0f, gyf);
    const int area = (o.rect[2] - o.rect[0]) * (o.rect[3] - o.rect[1]);
    if (area <= 0) return o;
    o.visible = true;
    o.tiles = (uint32_t)area;
    o.radius = (int)rf;
    o.mean2d[0] = m2x; o.mean2d[1] = m2y;
    std::memcpy(&o.depth_bits, &tf[2], 4);
    return o;
}

// ---------------------------------------------------------------------------------------------
// Small dense helpers (double)
// ---------------------------------------------------------------------------------------------
void quat_to_R(const double q[4], double R[3][3]) {
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0][0] = 1 - 2 * (y * y + z * z); R[0][1] = 2 * (x * y - w * z);     R[0][2] = 2 * (x * z + w * y);
    R[1][0] = 2 * (x * y + w * z);     R[1][1] = 1 - 2 * (x * x + z * z); R[1][2] = 2 * (y * z - w * x);
    R[2][0] = 2 * (x * z - w * y);     R[2][1] = 2 * (y * z + w * x);     R[2][2] = 1 - 2 * (x * x + y * y);
}

bool inv3(const double A[3][3], double B[3][3]) {
    const double c00 = A[1][1] * A[2][2] - A[1][2] * A[2][1];
    const double c01 = A[1][2] * A[2][0] - A[1][0] * A[2][2];
    const double c02 = A[1][0] * A[2][1] - A[1][1] * A[2][0];
    const double det = A[0][0] * c00 + A[0][1] * c01 + A[0][2] * c02;
    if (det == 0.0 || !std::isfinite(det)) return false;
    const double id = 1.0 / det;
    B[0][0] = c00 * id; B[1][0] = c01 * id; B[2][0] = c02 * id;
    B[0][1] = (A[0][2] * A[2][1] - A[0][1] * A[2][2]) * id;
    B[1][1] = (A[0][0] * A[2][2] - A[0][2] * A[2][0]) * id;
    B[2][1] = (A[0][1] * A[2][0] - A[0][0] * A[2][1]) * id;
    B[0][2] = (A[0][1] * A[1][2] - A[0][2] * A[1][1]) * id;
    B[1][2] = (A[0][2] * A[1][0] - A[0][0] * A[1][2]) * id;
    B[2][2] = (A[0][0] * A[1][1] - A[0][1] * A[1][0]) * id;
    return true;
}

// Real spherical harmonics to degree 3 (reading C22): values Y[16] and gradient dY[16][3] of the
// polynomial extension, at a unit direction d.
void sh_basis(const double d[3], double Y[16], double dY[16][3]) {
    const double PI = 3.14159265358979323846;
    const double k0 = std::sqrt(1.0 / (4 * PI)), k1 = std::sqrt(3.0 / (4 * PI));
    const double k2a = std::sqrt(15.0 / (4 * PI)), k2b = std::sqrt(5.0 / (16 * PI)), k2c = std::sqrt(15.0 / (16 * PI));
    const double k3a = std::sqrt(35.0 / (32 * PI)), k3b = std::sqrt(105.0 / (4 * PI)), k3c = std::sqrt(21.0 / (32 * PI));
    const double k3d = std::sqrt(7.0 / (16 * PI)), k3e = std::sqrt(105.0 / (16 * PI));
    const double x = d[0], y = d[1], z = d[2];
    const double xx = x * x, yy = y * y, zz = z * z;
    for (int j = 0; j < 16; ++j) dY[j][0] = dY[j][1] = dY[j][2] = 0.0;
    Y[0] = k0;
    Y[1] = -k1 * y;  dY[1][1] = -k1;
    Y[2] = k1 * z;   dY[2][2] = k1;
    Y[3] = -k1 * x;  dY[3][0] = -k1;
    Y[4] = k2a * x * y;   dY[4][0] = k2a * y;  dY[4][1] = k2a * x;
    Y[5] = -k2a * y * z;  dY[5][1] = -k2a * z; dY[5][2] = -k2a * y;
    Y[6] = k2b * (2 * zz - xx - yy); dY[6][0] = -2 * k2b * x; dY[6][1] = -2 * k2b * y; dY[6][2] = 4 * k2b * z;
    Y[7] = -k2a * x * z;  dY[7][0] = -k2a * z; dY[7][2] = -k2a * x;
    Y[8] = k2c * (xx - yy); dY[8][0] = 2 * k2c * x; dY[8][1] = -2 * k2c * y;
    Y[9] = -k3a * y * (3 * xx - yy);   dY[9][0] = -k3a * 6 * x * y;  dY[9][1] = -k3a * (3 * xx - 3 * yy);
    Y[10] = k3b * x * y * z;           dY[10][0] = k3b * y * z; dY[10][1] = k3b * x * z; dY[10][2] = k3b * x * y;
    Y[11] = -k3c * y * (4 * zz - xx - yy);
    dY[11][0] = k3c * 2 * x * y; dY[11][1] = -k3c * (4 * zz - xx - 3 * yy); dY[11][2] = -k3c * 8 * y * z;
    Y[12] = k3d * z * (2 * zz - 3 * xx - 3 * yy);
    dY[12][0] = -k3d * 6 * x * z; dY[12][1] = -k3d * 6 * y * z; dY[12][2] = k3d * (6 * zz - 3 * xx - 3 * yy);
    Y[13] = -k3c * x * (4 * zz - xx - yy);
    dY[13][0] = -k3c * (4 * zz - 3 * xx - yy); dY[13][1] = k3c * 2 * x * y; dY[13][2] = -k3c * 8 * x * z;
    Y[14] = k3e * z * (xx - yy);       dY[14][0] = k3e * 2 * x * z; dY[14][1] = -k3e * 2 * y * z; dY[14][2] = k3e * (xx - yy);
    Y[15] = -k3a * x * (xx - 3 * yy);  dY[15][0] = -k3a * (3 * xx - 3 * yy); dY[15][1] = k3a * 6 * x * y;
}

// ---------------------------------------------------------------------------------------------
// Projection of one primitive (values in double).  third_row selects the completion of J to 3x3
// used for the paper-literal frequency projection (reading C2): 0 -> (0,0,1); 1 -> t/|t| (EWA);
// 2 -> (0.3,-0.2,0.7).  f2D must not depend on it (pinned).
// ---------------------------------------------------------------------------------------------
struct Proj {
    Twin tw;
    double t[3], mean2d[2];
    double Sigma[3][3], J[2][3], T[2][3];
    bool clampx, clampy;
    double U[3];      // undilated U00, U01, U11
    double conic[3];  // a, b, c of (U + 0.3 I)^-1
    double f2d[KMAX][2];
    double rgb[3];
    bool clamped[3];
    double dir[3], vlen;
    // exposed for the pins of Eq.9-11 / Eq.16-17
    double A3[3][3], fproj[KMAX][3], Sig3[3][3];
    // variants (f4): att[k] = C2_k, computed for every primitive; att_used[k] = what the render multiplies w_k by
    // (C2_k or 1); rho = Mip opacity factor (1 without the variant); o_eff = o * rho
    double att[KMAX], att_used[KMAX], rho, o_eff, dilation;
};

void project_values(const Scene& s, const Cam& c, int i, int third_row, Proj& p) {
    const double mu[3] = {s.means[3 * i], s.means[3 * i + 1], s.means[3 * i + 2]};
    for (int a = 0; a < 3; ++a)
        p.t[a] = c.Wm[a][0] * mu[0] + c.Wm[a][1] * mu[1] + c.Wm[a][2] * mu[2] + c.tau[a];
    const double tz = p.t[2];
    // Sigma = R S S^T R^T
    const double q[4] = {s.quats[4 * i], s.quats[4 * i + 1], s.quats[4 * i + 2], s.quats[4 * i + 3]};
    double R[3][3];
    quat_to_R(q, R);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
        double v = 0;
        for (int k = 0; k < 3; ++k) { const double sk = s.scales[3 * i + k]; v += R[a][k] * sk * sk * R[b][k]; }
        p.Sigma[a][b] = v;
    }
    // J: Jacobian of (fx x/z, fy y/z) at the clamped ray direction (reading C8)
    const double limx = 1.3 * (0.5 * c.W / c.fx), limy = 1.3 * (0.5 * c.H / c.fy);
    double ux = p.t[0] / tz, uy = p.t[1] / tz;
    p.clampx = (ux < -limx) || (ux > limx);
    p.clampy = (uy < -limy) || (uy > limy);
    ux = std::min(limx, std::max(-limx, ux));
    uy = std::min(limy, std::max(-limy, uy));
    p.J[0][0] = c.fx / tz; p.J[0][1] = 0;         p.J[0][2] = -c.fx * ux / tz;
    p.J[1][0] = 0;         p.J[1][1] = c.fy / tz; p.J[1][2] = -c.fy * uy / tz;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 3; ++b)
        p.T[a][b] = p.J[a][0] * c.Wm[0][b] + p.J[a][1] * c.Wm[1][b] + p.J[a][2] * c.Wm[2][b];
    // Sigma' = J W Sigma W^T J^T, top-left 2x2                                      PAPER.md:91 Eq.2
    double V[2][3];
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 3; ++b)
        V[a][b] = p.T[a][0] * p.Sigma[0][b] + p.T[a][1] * p.Sigma[1][b] + p.T[a][2] * p.Sigma[2][b];
    p.U[0] = V[0][0] * p.T[0][0] + V[0][1] * p.T[0][1] + V[0][2] * p.T[0][2];
    p.U[1] = V[0][0] * p.T[1][0] + V[0][1] * p.T[1][1] + V[0][2] * p.T[1][2];
    p.U[2] = V[1][0] * p.T[1][0] + V[1][1] * p.T[1][1] + V[1][2] * p.T[1][2];
    // conic of the dilated 2D covariance                                            PAPER.md:101 Eq.3, reading C5
    p.dilation = (s.variant & VARIANT_MIP_FILTER) ? MIP_DILATION : DILATION;
    const double A = p.U[0] + p.dilation, B = p.U[1], C = p.U[2] + p.dilation;
    const double det = A * C - B * B;
    p.conic[0] = C / det; p.conic[1] = -B / det; p.conic[2] = A / det;
    // Mip filter: opacity factor sqrt(det U / det(U + 0.1 I))
    p.rho = (s.variant & VARIANT_MIP_FILTER) ? std::sqrt(std::max(0.0, (p.U[0] * p.U[2] - p.U[1] * p.U[1]) / det)) : 1.0;
    p.o_eff = (double)s.opac[i] * p.rho;
    // mu2D
    p.mean2d[0] = c.fx * p.t[0] / tz + c.cx;
    p.mean2d[1] = c.fy * p.t[1] / tz + c.cy;

    // Frequencies, literally as the paper writes them.                              PAPER.md:145 Eq.9, :414, :150-154 Eq.10-11
    double J3[3][3] = {{p.J[0][0], p.J[0][1], p.J[0][2]}, {p.J[1][0], p.J[1][1], p.J[1][2]}, {0, 0, 1}};
    if (third_row == 1) {
        const double l = std::sqrt(p.t[0] * p.t[0] + p.t[1] * p.t[1] + tz * tz);
        J3[2][0] = p.t[0] / l; J3[2][1] = p.t[1] / l; J3[2][2] = tz / l;
    } else if (third_row == 2) {
        J3[2][0] = 0.3; J3[2][1] = -0.2; J3[2][2] = 0.7;
    }
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
        p.A3[a][b] = J3[a][0] * c.Wm[0][b] + J3[a][1] * c.Wm[1][b] + J3[a][2] * c.Wm[2][b];
    double Ainv[3][3], AS[3][3], S[3][3];
    const bool okA = inv3(p.A3, Ainv);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
        AS[a][b] = p.A3[a][0] * p.Sigma[0][b] + p.A3[a][1] * p.Sigma[1][b] + p.A3[a][2] * p.Sigma[2][b];
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
        p.Sig3[a][b] = AS[a][0] * p.A3[b][0] + AS[a][1] * p.A3[b][1] + AS[a][2] * p.A3[b][2];
    const bool okS = inv3(p.Sig3, S);
    for (int k = 0; k < s.K; ++k) {
        const float* f = s.freqs + (size_t)(i * s.K + k) * 3;
        // f_proj^T = f^T (JW)^-1   <=>   f_proj = (JW)^-T f
        for (int a = 0; a < 3; ++a)
            p.fproj[k][a] = okA ? Ainv[0][a] * f[0] + Ainv[1][a] * f[1] + Ainv[2][a] * f[2] : 0.0;
        if (okA && okS) {
            p.f2d[k][0] = p.fproj[k][0] - S[0][2] / S[2][2] * p.fproj[k][2];            // Eq.10 / Eq.29
            p.f2d[k][1] = p.fproj[k][1] - S[1][2] / S[2][2] * p.fproj[k][2];
            p.att[k] = std::exp(-2.0 * (TWO_PI / 2) * (TWO_PI / 2) * p.fproj[k][2] * p.fproj[k][2] / S[2][2]);  // C2_k
        } else {
            p.f2d[k][0] = p.f2d[k][1] = 0.0;
            p.att[k] = 1.0;
        }
        p.att_used[k] = (s.variant & VARIANT_LINE_INTEGRAL) ? p.att[k] : 1.0;
    }
    // colour from SH at the viewing direction (reading C22, C8)
    double cam_pos[3];
    for (int a = 0; a < 3; ++a) cam_pos[a] = -(c.Wm[0][a] * c.tau[0] + c.Wm[1][a] * c.tau[1] + c.Wm[2][a] * c.tau[2]);
    double v[3] = {mu[0] - cam_pos[0], mu[1] - cam_pos[1], mu[2] - cam_pos[2]};
    p.vlen = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    for (int a = 0; a < 3; ++a) p.dir[a] = v[a] / p.vlen;
    double Y[16], dY[16][3];
    sh_basis(p.dir, Y, dY);
    const int ncoef = (s.deg + 1) * (s.deg + 1);
    for (int ch = 0; ch < 3; ++ch) {
        double acc = 0.5;
        for (int j = 0; j < ncoef; ++j) acc += Y[j] * s.sh[(size_t)i * 48 + j * 3 + ch];
        p.clamped[ch] = acc < 0.0;
        p.rgb[ch] = p.clamped[ch] ? 0.0 : acc;
    }
}

void project_all(const Scene& s, const Cam& c, int third_row, std::vector<Proj>& P) {
    P.resize(s.N);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < s.N; ++i) {
        P[i].tw = twin_index(s, c, i);
        if (P[i].tw.visible) project_values(s, c, i, third_row, P[i]);
    }
}

// Depth order: ascending (bits(float32 depth), primitive index)                      PAPER.md:103, readings C12-C13
std::vector<int> depth_order(const std::vector<Proj>& P) {
    std::vector<int> ord;
    for (int i = 0; i < (int)P.size(); ++i) if (P[i].tw.visible) ord.push_back(i);
    std::sort(ord.begin(), ord.end(), [&](int a, int b) {
        if (P[a].tw.depth_bits != P[b].tw.depth_bits) return P[a].tw.depth_bits < P[b].tw.depth_bits;
        return a < b;
    });
    return ord;
}

// ---------------------------------------------------------------------------------------------
// One primitive at one pixel: Eq.12 and the alpha rules (step 10 of DESIGN.md "Forward").
// ---------------------------------------------------------------------------------------------
struct PairEval {
    double dx, dy, G, M, raw, alpha;   // raw = o G M ; alpha = min(0.99, raw)
    double cosv[KMAX], sinv[KMAX];
    bool power_pos, envelope_pass;
};

inline void eval_pair(const Scene& s, const Proj& p, int i, double px, double py, PairEval& e) {
    e.dx = px - p.mean2d[0];
    e.dy = py - p.mean2d[1];
    const double q = -0.5 * (p.conic[0] * e.dx * e.dx + p.conic[2] * e.dy * e.dy) - p.conic[1] * e.dx * e.dy;  // Eq.3
    e.power_pos = q > 0.0;
    e.G = std::exp(q);
    const double o = p.o_eff;
    e.envelope_pass = o * e.G >= ALPHA_MIN;
    double wsum = 0.0, mod = 0.0;
    for (int k = 0; k < s.K; ++k) {
        const double w = s.weights[(size_t)i * s.K + k];
        const double phi = TWO_PI * (p.f2d[k][0] * e.dx + p.f2d[k][1] * e.dy);
        e.cosv[k] = std::cos(phi);
        e.sinv[k] = std::sin(phi);
        wsum += w;
        mod += w * p.att_used[k] * e.cosv[k];
    }
    e.M = (1.0 - wsum) + mod;                                                           // Eq.12 bracket
    e.raw = o * e.G * e.M;
    e.alpha = std::min(ALPHA_MAX, e.raw);
}

struct PixelState {
    double T = 1.0, C[3] = {0, 0, 0};
    bool done = false;
    uint32_t pos = 0, last_pos = 0;
    int32_t last_id = -1;
    uint32_t examined = 0, envelope = 0, blended = 0;
    double margin = 1e300, margin_clamp = 1e300;
    int32_t inj = -1;          // index into Inject (decision-injected mode), -1 = this pixel takes its own decisions
    uint32_t inj_at = 0;       // cursor into the pixel's injected list
};

// Decision-injected mode (reading C18).  The image is discontinuous where alpha crosses 1/255, where
// T (1 - alpha) crosses 1e-4 and (for the gradient) where o G M crosses 0.99: within the evaluation error of a
// threshold BOTH outcomes are correct renderings.  To compare gradients and images at such pixels without masking
// them, the caller may fix the outcome of every decision at selected pixels: for pixel pixels[i], the ascending
// 1-based tile-list positions of the entries that are blended (bit 31: the 0.99 clamp counts as active) and the
// position at which the pixel stops (0 = never).  The oracle evaluates every pair exactly as before, takes the
// injected outcome, and COUNTS A VIOLATION whenever the injected outcome differs from its own while its own value
// is farther than `delta` (relative) from the threshold concerned -- so an injected list is accepted only if it is a
// correct rendering in the sense above.  Pixels without an injected list are untouched.
struct Inject {
    int n = 0;
    const int32_t* pixels = nullptr;     // [n][2] (x, y)
    const uint32_t* offsets = nullptr;   // [n+1]
    const uint32_t* entries = nullptr;   // [offsets[n]]
    const uint32_t* stop_pos = nullptr;  // [n]
    double delta = 0.0;
    uint64_t* violations = nullptr;      // [1], incremented atomically
};

inline void violation(const Inject& inj) {
#pragma omp atomic
    inj.violations[0] += 1;
}

// Visit primitive i (already known to cover the pixel's tile) at pixel (px,py).
inline void visit_injected(const Scene& s, const Proj& p, int i, double px, double py, PixelState& st, const Inject& inj);

inline void visit(const Scene& s, const Proj& p, int i, double px, double py, PixelState& st, const Inject* inj = nullptr) {
    if (st.done) return;
    if (st.inj >= 0) { visit_injected(s, p, i, px, py, st, *inj); return; }
    st.pos += 1;
    st.examined += 1;
    PairEval e;
    eval_pair(s, p, i, px, py, e);
    if (e.power_pos) return;
    if (e.envelope_pass) st.envelope += 1;
    st.margin = std::min(st.margin, std::fabs(e.alpha - ALPHA_MIN) / ALPHA_MIN);
    if (e.alpha < ALPHA_MIN) return;
    st.margin_clamp = std::min(st.margin_clamp, std::fabs(e.raw - ALPHA_MAX) / ALPHA_MAX);
    const double Tn = st.T * (1.0 - e.alpha);
    st.margin = std::min(st.margin, std::fabs(Tn - T_MIN) / T_MIN);
    if (Tn < T_MIN) { st.done = true; return; }
    for (int ch = 0; ch < 3; ++ch) st.C[ch] += p.rgb[ch] * e.alpha * st.T;              // Eq.13
    st.T = Tn;
    st.last_pos = st.pos;
    st.last_id = i;
    st.blended += 1;
}

// The same visit with the outcome of every decision taken from the pixel's injected list (see Inject).
inline void visit_injected(const Scene& s, const Proj& p, int i, double px, double py, PixelState& st, const Inject& inj) {
    st.pos += 1;
    st.examined += 1;
    PairEval e;
    eval_pair(s, p, i, px, py, e);
    const uint32_t* lst = inj.entries + inj.offsets[st.inj];
    const uint32_t len = inj.offsets[st.inj + 1] - inj.offsets[st.inj];
    const bool take = st.inj_at < len && (lst[st.inj_at] & 0x7fffffffu) == st.pos;
    const bool stop_here = inj.stop_pos[st.inj] == st.pos;
    if (!e.power_pos && e.envelope_pass) st.envelope += 1;
    // the oracle's own outcome in the injected state: 0 skip, 1 stop, 2 blend
    const double Tn = st.T * (1.0 - e.alpha);
    const double m_alpha = std::fabs(e.alpha - ALPHA_MIN) / ALPHA_MIN;
    const double m_T = std::fabs(Tn - T_MIN) / T_MIN;
    const int own = (e.power_pos || e.alpha < ALPHA_MIN) ? 0 : (Tn < T_MIN ? 1 : 2);
    if (take) {
        if (stop_here) violation(inj);                                   // malformed list
        if (e.power_pos) violation(inj);
        else if (own == 0 && m_alpha > inj.delta) violation(inj);
        else if (own == 1 && m_T > inj.delta) violation(inj);
        const bool clamp = (lst[st.inj_at] >> 31) != 0;
        if (clamp != (e.raw > ALPHA_MAX) && std::fabs(e.raw - ALPHA_MAX) / ALPHA_MAX > inj.delta) violation(inj);
        st.inj_at += 1;
        for (int ch = 0; ch < 3; ++ch) st.C[ch] += p.rgb[ch] * e.alpha * st.T;              // Eq.13
        st.T = Tn;
        st.last_pos = st.pos;
        st.last_id = i;
        st.blended += 1;
        return;
    }
    if (stop_here) {
        // the pixel stops at this entry: correct iff its own outcome is "stop", or "blend" / "skip" within delta
        if (own == 2 && m_T > inj.delta) violation(inj);
        if (own == 0 && (e.power_pos || m_alpha > inj.delta)) violation(inj);
        if (st.inj_at != len) violation(inj);                            // blended entries listed after the stop
        st.done = true;
        return;
    }
    // skipped: correct iff its own outcome is "skip", or "blend" within delta of 1/255; a pixel that would stop
    // here on its own must also be within delta (the injected outcome says the walk goes on)
    if (own == 2 && m_alpha > inj.delta) violation(inj);
    if (own == 1 && m_alpha > inj.delta && m_T > inj.delta) violation(inj);
}

inline bool covers(const Twin& tw, int tx, int ty) {
    return tx >= tw.rect[0] && tx < tw.rect[2] && ty >= tw.rect[1] && ty < tw.rect[3];
}

struct FwdOut {
    double* image;      // [3][H][W]
    double* final_T;    // [H][W]
    uint32_t* n_contrib;  // [H][W] 1-based position in the tile list of the last blended primitive
    int32_t* last_id;   // [H][W]
    uint32_t* counters; // [H][W][3] examined, envelope-passing, blended
    double* margin;     // [H][W][2] forward decision margin, clamp margin
};

inline void store_pixel(const Cam& c, const FwdOut& o, int x, int y, const PixelState& st) {
    const size_t pix = (size_t)y * c.W + x, HW = (size_t)c.H * c.W;
    for (int ch = 0; ch < 3; ++ch) o.image[ch * HW + pix] = st.C[ch] + st.T * c.bg[ch];  // reading C23
    o.final_T[pix] = st.T;
    o.n_contrib[pix] = st.last_pos;
    o.last_id[pix] = st.last_id;
    if (o.counters) { o.counters[3 * pix] = st.examined; o.counters[3 * pix + 1] = st.envelope; o.counters[3 * pix + 2] = st.blended; }
    if (o.margin) { o.margin[2 * pix] = st.margin; o.margin[2 * pix + 1] = st.margin_clamp; }
}

// Painter's order, parallel over tile rows: primitive-major over the pixels of its rectangle.
void forward_painter(const Scene& s, const Cam& c, const std::vector<Proj>& P, const std::vector<int>& ord,
                     const FwdOut& out, std::vector<PixelState>* keep, const Inject* inj = nullptr) {
    std::vector<PixelState> local;
    std::vector<PixelState>& st = keep ? *keep : local;
    st.assign((size_t)c.W * c.H, PixelState());
    if (inj)
        for (int k = 0; k < inj->n; ++k) st[(size_t)inj->pixels[2 * k + 1] * c.W + inj->pixels[2 * k]].inj = k;
#pragma omp parallel for schedule(dynamic, 1)
    for (int ty = 0; ty < c.gy; ++ty) {
        const int y0 = ty * TILE, y1 = std::min(c.H, y0 + TILE);
        for (int i : ord) {
            const Twin& tw = P[i].tw;
            if (ty < tw.rect[1] || ty >= tw.rect[3]) continue;
            const int x0 = tw.rect[0] * TILE, x1 = std::min(c.W, tw.rect[2] * TILE);
            for (int y = y0; y < y1; ++y)
                for (int x = x0; x < x1; ++x) visit(s, P[i], i, (double)x, (double)y, st[(size_t)y * c.W + x], inj);
        }
        for (int y = y0; y < y1; ++y)
            for (int x = 0; x < c.W; ++x) {
                const PixelState& ps = st[(size_t)y * c.W + x];
                // an injected list must have been consumed entirely
                if (inj && ps.inj >= 0 && ps.inj_at != inj->offsets[ps.inj + 1] - inj->offsets[ps.inj]) violation(*inj);
                store_pixel(c, out, x, y, ps);
            }
    }
}

// ---------------------------------------------------------------------------------------------
// Backward.  dL/dC given; L = sum_p <g_C(p), C(p)>.  DESIGN.md "Backward" (derived; the paper
// gives no equations).  2D gradients per primitive:
// ---------------------------------------------------------------------------------------------
struct Grad2D {
    double rgb[3], o, conic[3], mean2d[2], f2d[KMAX][2], w[KMAX], absmean2d[2];
    double att[KMAX];   // dL/d att_used[k] (line-integral variant)
};

void backward_pixels(const Scene& s, const Cam& c, const std::vector<Proj>& P, const std::vector<int>& ord,
                     const std::vector<PixelState>& st, const float* gimg, std::vector<Grad2D>& G2,
                     const Inject* inj = nullptr) {
    const size_t HW = (size_t)c.H * c.W;
    G2.assign(s.N, Grad2D{});
    // position of each visible primitive in the depth order (for the "not beyond last" test)
#pragma omp parallel for schedule(dynamic, 1)
    for (int ty = 0; ty < c.gy; ++ty) {
        const int y0 = ty * TILE, y1 = std::min(c.H, y0 + TILE);
        // per-pixel reverse state: transmittance T (in front of the current primitive), B = colour behind
        std::vector<double> Tcur((size_t)TILE * c.W), Bc((size_t)TILE * c.W * 3);
        std::vector<uint32_t> pos((size_t)TILE * c.W);
        std::vector<uint32_t> icur((size_t)TILE * c.W, 0);   // injected pixels: entries of the list not yet walked
        if (inj)
            for (int y = y0; y < y1; ++y) for (int x = 0; x < c.W; ++x) {
                const int k = st[(size_t)y * c.W + x].inj;
                if (k >= 0) icur[(size_t)(y - y0) * c.W + x] = inj->offsets[k + 1] - inj->offsets[k];
            }
        // pos counts, per pixel, how many covering primitives remain (1-based position of the current one)
        for (int y = y0; y < y1; ++y) for (int x = 0; x < c.W; ++x) {
            const size_t l = (size_t)(y - y0) * c.W + x;
            Tcur[l] = st[(size_t)y * c.W + x].T;
            for (int ch = 0; ch < 3; ++ch) Bc[3 * l + ch] = c.bg[ch];
            pos[l] = 0;
        }
        // tile-list length per tile column of this row, to know each primitive's 1-based position walking back
        std::vector<uint32_t> len(c.gx, 0);
        for (int i : ord) { const Twin& tw = P[i].tw; if (ty >= tw.rect[1] && ty < tw.rect[3]) for (int tx = tw.rect[0]; tx < tw.rect[2]; ++tx) len[tx] += 1; }
        std::vector<uint32_t> cur(len);  // position of the primitive about to be visited, per tile column
        for (auto it = ord.rbegin(); it != ord.rend(); ++it) {
            const int i = *it;
            const Proj& p = P[i];
            const Twin& tw = p.tw;
            if (ty < tw.rect[1] || ty >= tw.rect[3]) continue;
            Grad2D acc{};
            for (int tx = tw.rect[0]; tx < tw.rect[2]; ++tx) {
                const uint32_t mypos = cur[tx];
                cur[tx] -= 1;
                const int x0 = tx * TILE, x1 = std::min(c.W, x0 + TILE);
                for (int y = y0; y < y1; ++y) for (int x = x0; x < x1; ++x) {
                    const PixelState& ps = st[(size_t)y * c.W + x];
                    if (mypos > ps.last_pos) continue;          // beyond the last blended primitive
                    const size_t l = (size_t)(y - y0) * c.W + x;
                    PairEval e;
                    bool clamp_active;
                    if (ps.inj >= 0) {
                        // decision-injected pixel: blended iff the position is the next one (from the back) of its list
                        if (icur[l] == 0) continue;
                        const uint32_t ent = inj->entries[inj->offsets[ps.inj] + icur[l] - 1];
                        if ((ent & 0x7fffffffu) != mypos) continue;
                        icur[l] -= 1;
                        eval_pair(s, p, i, (double)x, (double)y, e);
                        clamp_active = (ent >> 31) != 0;
                    } else {
                        eval_pair(s, p, i, (double)x, (double)y, e);
                        if (e.power_pos || e.alpha < ALPHA_MIN) continue;
                        clamp_active = e.raw > ALPHA_MAX;
                    }
                    const double Ti = Tcur[l] / (1.0 - e.alpha);   // transmittance in front of i
                    Tcur[l] = Ti;
                    const size_t pix = (size_t)y * c.W + x;
                    const double gC[3] = {gimg[pix], gimg[HW + pix], gimg[2 * HW + pix]};
                    double galpha = 0.0;
                    for (int ch = 0; ch < 3; ++ch) {
                        acc.rgb[ch] += e.alpha * Ti * gC[ch];
                        galpha += Ti * gC[ch] * (p.rgb[ch] - Bc[3 * l + ch]);
                        Bc[3 * l + ch] = e.alpha * p.rgb[ch] + (1.0 - e.alpha) * Bc[3 * l + ch];
                    }
                    if (clamp_active) continue;                  // clamp active: zero derivative (reading C14)
                    const double o = p.o_eff;
                    acc.o += galpha * e.G * e.M;                 // dL/d o_eff
                    const double gG = galpha * o * e.M, gM = galpha * o * e.G;
                    const double gq = gG * e.G;
                    double gdx = gq * (-p.conic[0] * e.dx - p.conic[1] * e.dy);
                    double gdy = gq * (-p.conic[2] * e.dy - p.conic[1] * e.dx);
                    acc.conic[0] += gq * (-0.5 * e.dx * e.dx);
                    acc.conic[1] += gq * (-e.dx * e.dy);
                    acc.conic[2] += gq * (-0.5 * e.dy * e.dy);
                    for (int k = 0; k < s.K; ++k) {
                        const double w = s.weights[(size_t)i * s.K + k];
                        acc.w[k] += gM * (p.att_used[k] * e.cosv[k] - 1.0);
                        acc.att[k] += gM * w * e.cosv[k];
                        const double gphi = -gM * w * p.att_used[k] * e.sinv[k];
                        acc.f2d[k][0] += gphi * TWO_PI * e.dx;
                        acc.f2d[k][1] += gphi * TWO_PI * e.dy;
                        gdx += gphi * TWO_PI * p.f2d[k][0];
                        gdy += gphi * TWO_PI * p.f2d[k][1];
                    }
                    acc.mean2d[0] -= gdx;
                    acc.mean2d[1] -= gdy;
                    acc.absmean2d[0] += std::fabs(gdx);
                    acc.absmean2d[1] += std::fabs(gdy);
                }
            }
            // accumulate this tile row's contribution (rows run in parallel)
            Grad2D& g = G2[i];
            double* dst = reinterpret_cast<double*>(&g);
            const double* src = reinterpret_cast<const double*>(&acc);
            for (size_t k = 0; k < sizeof(Grad2D) / sizeof(double); ++k) {
                if (src[k] != 0.0) {
#pragma omp atomic
                    dst[k] += src[k];
                }
            }
        }
    }
}

struct GradOut {
    double *d_means, *d_scales, *d_quats, *d_opac, *d_sh, *d_freqs, *d_weights;   // parameter gradients
    double *d_mean2d, *d_conic, *d_rgb, *d_freq2d, *d_absmean2d;                    // 2D gradients (stage checks)
};

// Chain rule 2D -> 3D for one primitive (per-primitive part).
void backward_primitive(const Scene& s, const Cam& c, const Proj& p, int i, const Grad2D& g, const GradOut& out) {
    const int K = s.K;
    // conic -> U :  Cm = Ud^-1,  G_U = -Cm Gc Cm, Gc = [[ga, gb/2],[gb/2, gc]]
    const double a = p.conic[0], b = p.conic[1], cc = p.conic[2];
    const double Gc[2][2] = {{g.conic[0], 0.5 * g.conic[1]}, {0.5 * g.conic[1], g.conic[2]}};
    const double Cm[2][2] = {{a, b}, {b, cc}};
    double tmp[2][2], GU[2][2];
    for (int r = 0; r < 2; ++r) for (int q = 0; q < 2; ++q) tmp[r][q] = Cm[r][0] * Gc[0][q] + Cm[r][1] * Gc[1][q];
    for (int r = 0; r < 2; ++r) for (int q = 0; q < 2; ++q) GU[r][q] = -(tmp[r][0] * Cm[0][q] + tmp[r][1] * Cm[1][q]);
    double gSigma[3][3] = {{0}}, gT[2][3] = {{0}};
    // f2D_k = U^-1 T Sigma f_k (U undilated; closed form of Eq.9-10, reading C2)
    const double Ud = p.U[0] * p.U[2] - p.U[1] * p.U[1];
    const double Ui[2][2] = {{p.U[2] / Ud, -p.U[1] / Ud}, {-p.U[1] / Ud, p.U[0] / Ud}};
    // Mip filter: o_eff = o rho, rho = sqrt(det U / det U_d):  d rho = rho/2 tr((U^-1 - U_d^-1) dU)
    double g_opacity = g.o;
    if (s.variant & VARIANT_MIP_FILTER) {
        g_opacity = g.o * p.rho;
        const double grho = g.o * (double)s.opac[i];
        for (int r = 0; r < 2; ++r) for (int q = 0; q < 2; ++q) GU[r][q] += grho * p.rho * 0.5 * (Ui[r][q] - Cm[r][q]);
    }
    // line-integral attenuation: att_k = exp(-2 pi^2 a_k^2 / b), a_k = v . f_k, b = v^T Sigma^-1 v, where v spans the
    // null space of T = J W (the world-space direction of the ray): (f_z'')^2 / S22 = (v.f)^2 / (v^T Sigma^-1 v) for
    // any completion of J (reading C2); v = W^T (u_x, u_y, 1), (u_x, u_y) the clamped ray direction of J.
    double g_freq_extra[KMAX][3] = {{0}};
    double gt_extra[3] = {0, 0, 0};
    if ((s.variant & VARIANT_LINE_INTEGRAL) && K > 0) {
        const double tz0 = p.t[2];
        const double lx = 1.3 * (0.5 * c.W / c.fx), ly = 1.3 * (0.5 * c.H / c.fy);
        const double cdir[3] = {std::min(lx, std::max(-lx, p.t[0] / tz0)), std::min(ly, std::max(-ly, p.t[1] / tz0)), 1.0};
        double v[3], y[3];
        for (int m = 0; m < 3; ++m) v[m] = c.Wm[0][m] * cdir[0] + c.Wm[1][m] * cdir[1] + c.Wm[2][m] * cdir[2];
        double Si[3][3];
        inv3(p.Sigma, Si);
        for (int m = 0; m < 3; ++m) y[m] = Si[m][0] * v[0] + Si[m][1] * v[1] + Si[m][2] * v[2];
        const double b = v[0] * y[0] + v[1] * y[1] + v[2] * y[2];
        double gv[3] = {0, 0, 0}, gb = 0.0;
        const double PI2 = (TWO_PI / 2) * (TWO_PI / 2);
        for (int k = 0; k < K; ++k) {
            const float* f = s.freqs + (size_t)(i * K + k) * 3;
            const double a = v[0] * f[0] + v[1] * f[1] + v[2] * f[2];
            const double gatt = g.att[k] * p.att[k];                       // dL/d(ln att_k)
            const double ga = gatt * (-4.0 * PI2 * a / b);
            gb += gatt * (2.0 * PI2 * a * a / (b * b));
            for (int m = 0; m < 3; ++m) { g_freq_extra[k][m] = ga * v[m]; gv[m] += ga * f[m]; }
        }
        for (int m = 0; m < 3; ++m) gv[m] += gb * 2.0 * y[m];
        for (int m = 0; m < 3; ++m) for (int n = 0; n < 3; ++n) gSigma[m][n] -= gb * y[m] * y[n];   // d(Sigma^-1) = -Sigma^-1 dSigma Sigma^-1
        double gc[3];
        for (int a = 0; a < 3; ++a) gc[a] = c.Wm[a][0] * gv[0] + c.Wm[a][1] * gv[1] + c.Wm[a][2] * gv[2];
        if (!p.clampx) { gt_extra[0] += gc[0] / tz0; gt_extra[2] -= gc[0] * p.t[0] / (tz0 * tz0); }
        if (!p.clampy) { gt_extra[1] += gc[1] / tz0; gt_extra[2] -= gc[1] * p.t[1] / (tz0 * tz0); }
    }
    for (int k = 0; k < K; ++k) {
        const float* f = s.freqs + (size_t)(i * K + k) * 3;
        const double gf[2] = {g.f2d[k][0], g.f2d[k][1]};
        const double h[2] = {Ui[0][0] * gf[0] + Ui[0][1] * gf[1], Ui[1][0] * gf[0] + Ui[1][1] * gf[1]};
        const double* fk = p.f2d[k];
        for (int r = 0; r < 2; ++r) for (int q = 0; q < 2; ++q) GU[r][q] -= 0.5 * (h[r] * fk[q] + fk[r] * h[q]);
        double Th[3], Sf[3];
        for (int m = 0; m < 3; ++m) Th[m] = p.T[0][m] * h[0] + p.T[1][m] * h[1];
        for (int m = 0; m < 3; ++m) Sf[m] = p.Sigma[m][0] * f[0] + p.Sigma[m][1] * f[1] + p.Sigma[m][2] * f[2];
        for (int m = 0; m < 3; ++m) for (int n = 0; n < 3; ++n) gSigma[m][n] += 0.5 * (Th[m] * f[n] + f[m] * Th[n]);
        for (int r = 0; r < 2; ++r) for (int m = 0; m < 3; ++m) gT[r][m] += h[r] * Sf[m];
        for (int m = 0; m < 3; ++m)
            out.d_freqs[(size_t)(i * K + k) * 3 + m] = p.Sigma[m][0] * Th[0] + p.Sigma[m][1] * Th[1] + p.Sigma[m][2] * Th[2] + g_freq_extra[k][m];
        out.d_weights[(size_t)i * K + k] = g.w[k];
    }
    // U = T Sigma T^T
    double GUT[2][3];
    for (int r = 0; r < 2; ++r) for (int m = 0; m < 3; ++m) GUT[r][m] = GU[r][0] * p.T[0][m] + GU[r][1] * p.T[1][m];
    for (int m = 0; m < 3; ++m) for (int n = 0; n < 3; ++n) gSigma[m][n] += p.T[0][m] * GUT[0][n] + p.T[1][m] * GUT[1][n];
    for (int r = 0; r < 2; ++r) for (int m = 0; m < 3; ++m)
        gT[r][m] += 2.0 * (GUT[r][0] * p.Sigma[0][m] + GUT[r][1] * p.Sigma[1][m] + GUT[r][2] * p.Sigma[2][m]);
    // T = J W  ->  g_J = g_T W^T
    double gJ[2][3];
    for (int r = 0; r < 2; ++r) for (int m = 0; m < 3; ++m)
        gJ[r][m] = gT[r][0] * c.Wm[m][0] + gT[r][1] * c.Wm[m][1] + gT[r][2] * c.Wm[m][2];
    // J(t) and mu2D(t)
    const double tx = p.t[0], ty = p.t[1], tz = p.t[2];
    const double limx = 1.3 * (0.5 * c.W / c.fx), limy = 1.3 * (0.5 * c.H / c.fy);
    const double ux = std::min(limx, std::max(-limx, tx / tz)), uy = std::min(limy, std::max(-limy, ty / tz));
    double gt[3] = {gt_extra[0], gt_extra[1], gt_extra[2]};
    gt[2] += gJ[0][0] * (-c.fx / (tz * tz)) + gJ[1][1] * (-c.fy / (tz * tz));
    gt[2] += gJ[0][2] * (c.fx * ux / (tz * tz)) + gJ[1][2] * (c.fy * uy / (tz * tz));
    if (!p.clampx) { gt[0] += gJ[0][2] * (-c.fx / (tz * tz)); gt[2] += gJ[0][2] * (c.fx * tx / (tz * tz * tz)); }
    if (!p.clampy) { gt[1] += gJ[1][2] * (-c.fy / (tz * tz)); gt[2] += gJ[1][2] * (c.fy * ty / (tz * tz * tz)); }
    gt[0] += g.mean2d[0] * c.fx / tz;
    gt[1] += g.mean2d[1] * c.fy / tz;
    gt[2] += -g.mean2d[0] * c.fx * tx / (tz * tz) - g.mean2d[1] * c.fy * ty / (tz * tz);
    double gmu[3];
    for (int m = 0; m < 3; ++m) gmu[m] = c.Wm[0][m] * gt[0] + c.Wm[1][m] * gt[1] + c.Wm[2][m] * gt[2];
    // Sigma = Ms Ms^T, Ms = R diag(s)
    const double q[4] = {s.quats[4 * i], s.quats[4 * i + 1], s.quats[4 * i + 2], s.quats[4 * i + 3]};
    double R[3][3];
    quat_to_R(q, R);
    double gMs[3][3], gR[3][3];
    for (int m = 0; m < 3; ++m) for (int n = 0; n < 3; ++n) {
        double v = 0;
        for (int l = 0; l < 3; ++l) v += 2.0 * gSigma[m][l] * R[l][n] * s.scales[3 * i + n];
        gMs[m][n] = v;
    }
    for (int n = 0; n < 3; ++n) {
        double v = 0;
        for (int m = 0; m < 3; ++m) { v += R[m][n] * gMs[m][n]; gR[m][n] = gMs[m][n] * s.scales[3 * i + n]; }
        out.d_scales[3 * i + n] = v;
    }
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    out.d_quats[4 * i + 0] = 2 * (-z * gR[0][1] + y * gR[0][2] + z * gR[1][0] - x * gR[1][2] - y * gR[2][0] + x * gR[2][1]);
    out.d_quats[4 * i + 1] = 2 * (y * gR[0][1] + z * gR[0][2] + y * gR[1][0] - 2 * x * gR[1][1] - w * gR[1][2] + z * gR[2][0] + w * gR[2][1] - 2 * x * gR[2][2]);
    out.d_quats[4 * i + 2] = 2 * (-2 * y * gR[0][0] + x * gR[0][1] + w * gR[0][2] + x * gR[1][0] + z * gR[1][2] - w * gR[2][0] + z * gR[2][1] - 2 * y * gR[2][2]);
    out.d_quats[4 * i + 3] = 2 * (-2 * z * gR[0][0] - w * gR[0][1] + x * gR[0][2] + w * gR[1][0] - 2 * z * gR[1][1] + y * gR[1][2] + x * gR[2][0] + y * gR[2][1]);
    // colour: rgb = max(0, 0.5 + sum_j Y_j(dir) sh_j)
    double Y[16], dY[16][3];
    sh_basis(p.dir, Y, dY);
    const int ncoef = (s.deg + 1) * (s.deg + 1);
    double gdir[3] = {0, 0, 0};
    for (int ch = 0; ch < 3; ++ch) {
        const double gr = p.clamped[ch] ? 0.0 : g.rgb[ch];
        for (int j = 0; j < ncoef; ++j) {
            out.d_sh[(size_t)i * 48 + j * 3 + ch] = Y[j] * gr;
            const double shv = s.sh[(size_t)i * 48 + j * 3 + ch];
            for (int m = 0; m < 3; ++m) gdir[m] += dY[j][m] * shv * gr;
        }
    }
    const double dg = p.dir[0] * gdir[0] + p.dir[1] * gdir[1] + p.dir[2] * gdir[2];
    for (int m = 0; m < 3; ++m) gmu[m] += (gdir[m] - p.dir[m] * dg) / p.vlen;
    for (int m = 0; m < 3; ++m) out.d_means[3 * i + m] = gmu[m];
    out.d_opac[i] = g_opacity;
}

// deg carries the SH degree in its low byte and the variant flags in the next one (the C interface keeps one
// argument list for every entry point)
Scene make_scene(int N, int K, int deg, const float* means, const float* scales, const float* quats,
                 const float* opac, const float* sh, const float* freqs, const float* weights) {
    return Scene{N, K, deg & 0xff, means, scales, quats, opac, sh, freqs, weights, (deg >> 8) & 0xff};
}

}  // namespace

#define SCENE_ARGS int N, int K, int deg, const float* means, const float* scales, const float* quats, \
                   const float* opac, const float* sh, const float* freqs, const float* weights
#define SCENE_PASS N, K, deg, means, scales, quats, opac, sh, freqs, weights

extern "C" {

int orc_max_threads() { return omp_get_max_threads(); }
void orc_set_threads(int n) { if (n > 0) omp_set_num_threads(n); }

// Real SH basis (reading C22) at n unit directions: Y[n][16], dY[n][16][3].  Exposed for its pins.
void orc_sh_basis(int n, const double* dirs, double* Y, double* dY) {
    for (int k = 0; k < n; ++k) {
        double y[16], dy[16][3];
        sh_basis(dirs + 3 * k, y, dy);
        for (int j = 0; j < 16; ++j) {
            Y[16 * k + j] = y[j];
            for (int a = 0; a < 3; ++a) dY[(size_t)(16 * k + j) * 3 + a] = dy[j][a];
        }
    }
}

// Per-primitive projection outputs.  Any output pointer may be null.
void orc_project(SCENE_ARGS, const double* cam, int third_row,
                 uint8_t* visible, double* t, double* mean2d, double* cov2d, double* conic, double* freq2d,
                 double* rgb, uint8_t* clamped, uint32_t* depth_bits, float* mean2d_f32, int32_t* radius,
                 int32_t* rect, uint32_t* tiles_touched, double* A3, double* fproj, double* Sigma3,
                 double* att, double* rho) {
    const Scene s = make_scene(SCENE_PASS);
    const Cam c = load_cam(cam);
    std::vector<Proj> P;
    project_all(s, c, third_row, P);
    for (int i = 0; i < N; ++i) {
        const Proj& p = P[i];
        const bool v = p.tw.visible;
        if (visible) visible[i] = v;
        if (depth_bits) depth_bits[i] = v ? p.tw.depth_bits : 0;
        if (radius) radius[i] = v ? p.tw.radius : 0;
        if (tiles_touched) tiles_touched[i] = v ? p.tw.tiles : 0;
        for (int a = 0; a < 4; ++a) if (rect) rect[4 * i + a] = v ? p.tw.rect[a] : 0;
        for (int a = 0; a < 2; ++a) if (mean2d_f32) mean2d_f32[2 * i + a] = v ? p.tw.mean2d[a] : 0.f;
        for (int a = 0; a < 3; ++a) {
            if (t) t[3 * i + a] = v ? p.t[a] : 0;
            if (cov2d) cov2d[3 * i + a] = v ? p.U[a] : 0;
            if (conic) conic[3 * i + a] = v ? p.conic[a] : 0;
            if (rgb) rgb[3 * i + a] = v ? p.rgb[a] : 0;
            if (clamped) clamped[3 * i + a] = v ? p.clamped[a] : 0;
        }
        for (int a = 0; a < 2; ++a) if (mean2d) mean2d[2 * i + a] = v ? p.mean2d[a] : 0;
        for (int k = 0; k < K; ++k) {
            for (int a = 0; a < 2; ++a) if (freq2d) freq2d[(size_t)(i * K + k) * 2 + a] = v ? p.f2d[k][a] : 0;
            for (int a = 0; a < 3; ++a) if (fproj) fproj[(size_t)(i * K + k) * 3 + a] = v ? p.fproj[k][a] : 0;
            if (att) att[(size_t)i * K + k] = v ? p.att[k] : 0;
        }
        if (rho) rho[i] = v ? p.rho : 0;
        for (int a = 0; a < 9; ++a) {
            if (A3) A3[9 * i + a] = v ? p.A3[a / 3][a % 3] : 0;
            if (Sigma3) Sigma3[9 * i + a] = v ? p.Sig3[a / 3][a % 3] : 0;
        }
    }
}

// Tile lists.  mode 0: brute force, tile-major (for each tile, every primitive whose rectangle
// contains it, sorted by (depth bits, index)).  mode 1: emit (key, id) primitive-major, row-major over
// the rectangle, then std::stable_sort by key (feasible at full size).  Returns the instance count;
// fills the outputs only if capacity suffices.  key = (tile << 32) | depth_bits.
uint64_t orc_bin(SCENE_ARGS, const double* cam, int mode, uint64_t capacity,
                 uint64_t* keys, uint32_t* ids, uint32_t* ranges) {
    const Scene s = make_scene(SCENE_PASS);
    const Cam c = load_cam(cam);
    std::vector<Twin> tw(N);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) tw[i] = twin_index(s, c, i);
    uint64_t D = 0;
    for (int i = 0; i < N; ++i) if (tw[i].visible) D += tw[i].tiles;
    if (D > capacity || !keys) return D;
    const int ntiles = c.gx * c.gy;
    if (mode == 0) {
        uint64_t at = 0;
        for (int tile = 0; tile < ntiles; ++tile) {
            const int tx = tile % c.gx, ty = tile / c.gx;
            std::vector<std::pair<uint32_t, uint32_t>> lst;
            for (int i = 0; i < N; ++i) if (tw[i].visible && covers(tw[i], tx, ty)) lst.push_back({tw[i].depth_bits, (uint32_t)i});
            std::sort(lst.begin(), lst.end());
            ranges[2 * tile] = (uint32_t)at;
            for (auto& e : lst) { keys[at] = ((uint64_t)tile << 32) | e.first; ids[at] = e.second; ++at; }
            ranges[2 * tile + 1] = (uint32_t)at;
        }
    } else {
        std::vector<std::pair<uint64_t, uint32_t>> inst;
        inst.reserve(D);
        for (int i = 0; i < N; ++i) if (tw[i].visible)
            for (int ty = tw[i].rect[1]; ty < tw[i].rect[3]; ++ty)
                for (int tx = tw[i].rect[0]; tx < tw[i].rect[2]; ++tx)
                    inst.push_back({((uint64_t)(ty * c.gx + tx) << 32) | tw[i].depth_bits, (uint32_t)i});
        std::stable_sort(inst.begin(), inst.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
        for (int tile = 0; tile < ntiles; ++tile) ranges[2 * tile] = ranges[2 * tile + 1] = 0;
        for (uint64_t k = 0; k < D; ++k) {
            keys[k] = inst[k].first; ids[k] = inst[k].second;
            const uint32_t tile = (uint32_t)(inst[k].first >> 32);
            if (k == 0 || (uint32_t)(inst[k - 1].first >> 32) != tile) ranges[2 * tile] = (uint32_t)k;
            if (k + 1 == D || (uint32_t)(inst[k + 1].first >> 32) != tile) ranges[2 * tile + 1] = (uint32_t)(k + 1);
        }
    }
    return D;
}

// Forward render.  literal != 0: pixel-major loop over ALL primitives in depth order (O(N W H), tiny
// scenes only); literal == 0: painter's order (identical per-pixel arithmetic sequence).
void orc_render_forward(SCENE_ARGS, const double* cam, int literal, double* image, double* final_T,
                        uint32_t* n_contrib, int32_t* last_id, uint32_t* counters, double* margin) {
    const Scene s = make_scene(SCENE_PASS);
    const Cam c = load_cam(cam);
    std::vector<Proj> P;
    project_all(s, c, 0, P);
    const std::vector<int> ord = depth_order(P);
    const FwdOut out{image, final_T, n_contrib, last_id, counters, margin};
    if (!literal) { forward_painter(s, c, P, ord, out, nullptr); return; }
#pragma omp parallel for schedule(dynamic, 16)
    for (int y = 0; y < c.H; ++y)
        for (int x = 0; x < c.W; ++x) {
            PixelState st;
            for (int i : ord) if (covers(P[i].tw, x / TILE, y / TILE)) visit(s, P[i], i, (double)x, (double)y, st);
            store_pixel(c, out, x, y, st);
        }
}

// Auxiliary renders (the paper's frequency-map diagnostic): the same compositing
// (Eq.12-13, same lists, same alpha rules) with the colour of primitive i replaced by
//   ( sum_k omega_k |f2D_k|  [cycles per pixel],   t_z  [camera depth],   1 )
// over a zero background: channel 0 is the blended frequency map, channel 1 the blended depth, channel 2 the
// accumulated alpha (= 1 - final T).
void orc_render_aux(SCENE_ARGS, const double* cam, double* image, double* final_T) {
    const Scene s = make_scene(SCENE_PASS);
    Cam c = load_cam(cam);
    c.bg[0] = c.bg[1] = c.bg[2] = 0.0;
    std::vector<Proj> P;
    project_all(s, c, 0, P);
    for (int i = 0; i < N; ++i) {
        Proj& p = P[i];
        if (!p.tw.visible) continue;
        double fm = 0.0;
        for (int k = 0; k < K; ++k) fm += (double)s.weights[(size_t)i * K + k] * std::sqrt(p.f2d[k][0] * p.f2d[k][0] + p.f2d[k][1] * p.f2d[k][1]);
        p.rgb[0] = fm; p.rgb[1] = p.t[2]; p.rgb[2] = 1.0;
    }
    const std::vector<int> ord = depth_order(P);
    std::vector<uint32_t> nc((size_t)c.W * c.H), cnt((size_t)c.W * c.H * 3);
    std::vector<int32_t> last((size_t)c.W * c.H);
    std::vector<double> margin((size_t)c.W * c.H * 2);
    const FwdOut out{image, final_T, nc.data(), last.data(), cnt.data(), margin.data()};
    forward_painter(s, c, P, ord, out, nullptr);
}

// Literal render of selected pixels only (full-size spot checks).  pixels = [n][2] (x, y).
// Outputs are per selected pixel: colour[n][3], final_T[n], n_contrib[n], last_id[n], margin[n][2].
void orc_render_pixels(SCENE_ARGS, const double* cam, int n, const int32_t* pixels, double* colour,
                       double* final_T, uint32_t* n_contrib, int32_t* last_id, double* margin) {
    const Scene s = make_scene(SCENE_PASS);
    const Cam c = load_cam(cam);
    std::vector<Proj> P;
    project_all(s, c, 0, P);
    const std::vector<int> ord = depth_order(P);
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n; ++k) {
        const int x = pixels[2 * k], y = pixels[2 * k + 1];
        PixelState st;
        for (int i : ord) if (covers(P[i].tw, x / TILE, y / TILE)) visit(s, P[i], i, (double)x, (double)y, st);
        for (int ch = 0; ch < 3; ++ch) colour[3 * k + ch] = st.C[ch] + st.T * c.bg[ch];
        final_T[k] = st.T; n_contrib[k] = st.last_pos; last_id[k] = st.last_id;
        margin[2 * k] = st.margin; margin[2 * k + 1] = st.margin_clamp;
    }
}

// The oracle's own decisions at selected pixels, in the format of Inject: for pixel k the ascending 1-based
// tile-list positions of the entries it blends (bit 31: o G M > 0.99, clamp active) written to
// entries[offsets[k] .. offsets[k+1]) (dropped beyond the slice), counts[k] = number blended, stop_pos[k] = position
// of the entry at which T (1 - alpha) < 1e-4 stopped the pixel (0 = never).
void orc_trace_pixels(SCENE_ARGS, const double* cam, int n, const int32_t* pixels, const uint32_t* offsets,
                      uint32_t* entries, uint32_t* counts, uint32_t* stop_pos) {
    const Scene s = make_scene(SCENE_PASS);
    const Cam c = load_cam(cam);
    std::vector<Proj> P;
    project_all(s, c, 0, P);
    const std::vector<int> ord = depth_order(P);
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n; ++k) {
        const int x = pixels[2 * k], y = pixels[2 * k + 1];
        PixelState st;
        uint32_t nb = 0, stop = 0;
        const uint32_t cap = offsets[k + 1] - offsets[k];
        for (int i : ord) {
            if (!covers(P[i].tw, x / TILE, y / TILE)) continue;
            const uint32_t before = st.blended;
            visit(s, P[i], i, (double)x, (double)y, st);
            if (st.blended != before) {
                PairEval e;
                eval_pair(s, P[i], i, (double)x, (double)y, e);
                if (nb < cap) entries[offsets[k] + nb] = st.pos | (e.raw > ALPHA_MAX ? 0x80000000u : 0u);
                ++nb;
            }
            if (st.done) { stop = st.pos; break; }
        }
        counts[k] = nb;
        stop_pos[k] = stop;
    }
}

// Forward + analytic backward.  dL_dimage is [3][H][W] float32.  Gradient outputs are double, fully
// overwritten (zero for culled primitives).  The 2D-gradient outputs, final_T and n_contrib may be null.
// n_inj > 0 selects the decision-injected mode (see Inject): inj_pixels [n_inj][2], inj_offsets [n_inj+1],
// inj_entries, inj_stop [n_inj], accepted within the relative margin inj_delta; *violations counts the injected
// outcomes that are NOT correct renderings.
void orc_render_backward_ex(SCENE_ARGS, const double* cam, const float* dL_dimage, double* image, double* final_T,
                            uint32_t* n_contrib,
                            double* d_means, double* d_scales, double* d_quats, double* d_opac, double* d_sh,
                            double* d_freqs, double* d_weights, double* d_mean2d, double* d_conic, double* d_rgb,
                            double* d_freq2d, double* d_absmean2d,
                            int n_inj, const int32_t* inj_pixels, const uint32_t* inj_offsets, const uint32_t* inj_entries,
                            const uint32_t* inj_stop, double inj_delta, uint64_t* violations) {
    const Scene s = make_scene(SCENE_PASS);
    const Cam c = load_cam(cam);
    std::vector<Proj> P;
    project_all(s, c, 0, P);
    const std::vector<int> ord = depth_order(P);
    const size_t HW = (size_t)c.W * c.H;
    std::vector<double> img(3 * HW), fT(HW);
    std::vector<uint32_t> nc(HW);
    std::vector<int32_t> lid(HW);
    std::vector<PixelState> st;
    Inject inj;
    uint64_t dummy = 0;
    if (n_inj > 0) {
        inj.n = n_inj; inj.pixels = inj_pixels; inj.offsets = inj_offsets; inj.entries = inj_entries;
        inj.stop_pos = inj_stop; inj.delta = inj_delta; inj.violations = violations ? violations : &dummy;
        inj.violations[0] = 0;
    }
    const Inject* ip = n_inj > 0 ? &inj : nullptr;
    forward_painter(s, c, P, ord, FwdOut{img.data(), fT.data(), nc.data(), lid.data(), nullptr, nullptr}, &st, ip);
    if (image) std::memcpy(image, img.data(), 3 * HW * sizeof(double));
    if (final_T) std::memcpy(final_T, fT.data(), HW * sizeof(double));
    if (n_contrib) std::memcpy(n_contrib, nc.data(), HW * sizeof(uint32_t));
    std::vector<Grad2D> G2;
    backward_pixels(s, c, P, ord, st, dL_dimage, G2, ip);
    const GradOut out{d_means, d_scales, d_quats, d_opac, d_sh, d_freqs, d_weights, d_mean2d, d_conic, d_rgb, d_freq2d, d_absmean2d};
    std::memset(d_means, 0, sizeof(double) * 3 * N); std::memset(d_scales, 0, sizeof(double) * 3 * N);
    std::memset(d_quats, 0, sizeof(double) * 4 * N); std::memset(d_opac, 0, sizeof(double) * N);
    std::memset(d_sh, 0, sizeof(double) * 48 * N);
    std::memset(d_freqs, 0, sizeof(double) * 3 * (size_t)N * K); std::memset(d_weights, 0, sizeof(double) * (size_t)N * K);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        const Grad2D& g = G2[i];
        for (int a = 0; a < 2; ++a) {
            if (d_mean2d) d_mean2d[2 * i + a] = g.mean2d[a];
            if (d_absmean2d) d_absmean2d[2 * i + a] = g.absmean2d[a];
        }
        for (int a = 0; a < 3; ++a) { if (d_conic) d_conic[3 * i + a] = g.conic[a]; if (d_rgb) d_rgb[3 * i + a] = g.rgb[a]; }
        for (int k = 0; k < K; ++k) for (int a = 0; a < 2; ++a) if (d_freq2d) d_freq2d[(size_t)(i * K + k) * 2 + a] = g.f2d[k][a];
        if (P[i].tw.visible) backward_primitive(s, c, P[i], i, g, out);
    }
}

void orc_render_backward(SCENE_ARGS, const double* cam, const float* dL_dimage, double* image,
                         double* d_means, double* d_scales, double* d_quats, double* d_opac, double* d_sh,
                         double* d_freqs, double* d_weights, double* d_mean2d, double* d_conic, double* d_rgb,
                         double* d_freq2d, double* d_absmean2d) {
    orc_render_backward_ex(SCENE_PASS, cam, dL_dimage, image, nullptr, nullptr, d_means, d_scales, d_quats, d_opac, d_sh,
                           d_freqs, d_weights, d_mean2d, d_conic, d_rgb, d_freq2d, d_absmean2d, 0, nullptr, nullptr, nullptr,
                           nullptr, 0.0, nullptr);
}

}  // extern "C"
