// Real spherical harmonics to degree 3 (orthonormal on the sphere; order and signs of DESIGN.md reading
// C22): values and the gradient of their polynomial extension.  Device code of the CUDA path only.
#pragma once

namespace gabsplat {

// sqrt(1/4pi), sqrt(3/4pi), sqrt(15/4pi), sqrt(5/16pi), sqrt(15/16pi),
// sqrt(35/32pi), sqrt(105/4pi), sqrt(21/32pi), sqrt(7/16pi), sqrt(105/16pi)
#define GS_SH_C0 0.28209479177387814
#define GS_SH_C1 0.4886025119029199
#define GS_SH_C2A 1.0925484305920792
#define GS_SH_C2B 0.31539156525252005
#define GS_SH_C2C 0.5462742152960396
#define GS_SH_C3A 0.5900435899266435
#define GS_SH_C3B 2.890611442640554
#define GS_SH_C3C 0.4570457994644658
#define GS_SH_C3D 0.3731763325901154
#define GS_SH_C3E 1.445305721320277

// Y[j], j < (deg+1)^2, at the unit direction (x,y,z).
__device__ __forceinline__ void sh_values(int deg, double x, double y, double z, double* Y) {
  Y[0] = GS_SH_C0;
  if (deg < 1) return;
  Y[1] = -GS_SH_C1 * y;
  Y[2] = GS_SH_C1 * z;
  Y[3] = -GS_SH_C1 * x;
  if (deg < 2) return;
  const double xx = x * x, yy = y * y, zz = z * z;
  Y[4] = GS_SH_C2A * x * y;
  Y[5] = -GS_SH_C2A * y * z;
  Y[6] = GS_SH_C2B * (2.0 * zz - xx - yy);
  Y[7] = -GS_SH_C2A * x * z;
  Y[8] = GS_SH_C2C * (xx - yy);
  if (deg < 3) return;
  Y[9] = -GS_SH_C3A * y * (3.0 * xx - yy);
  Y[10] = GS_SH_C3B * x * y * z;
  Y[11] = -GS_SH_C3C * y * (4.0 * zz - xx - yy);
  Y[12] = GS_SH_C3D * z * (2.0 * zz - 3.0 * xx - 3.0 * yy);
  Y[13] = -GS_SH_C3C * x * (4.0 * zz - xx - yy);
  Y[14] = GS_SH_C3E * z * (xx - yy);
  Y[15] = -GS_SH_C3A * x * (xx - 3.0 * yy);
}

// dY[j][a] = d Y_j / d (x,y,z)_a of the polynomial extension, j < (deg+1)^2.
__device__ __forceinline__ void sh_gradients(int deg, double x, double y, double z, double (*dY)[3]) {
  dY[0][0] = dY[0][1] = dY[0][2] = 0.0;
  if (deg < 1) return;
  dY[1][0] = 0.0; dY[1][1] = -GS_SH_C1; dY[1][2] = 0.0;
  dY[2][0] = 0.0; dY[2][1] = 0.0; dY[2][2] = GS_SH_C1;
  dY[3][0] = -GS_SH_C1; dY[3][1] = 0.0; dY[3][2] = 0.0;
  if (deg < 2) return;
  const double xx = x * x, yy = y * y, zz = z * z;
  dY[4][0] = GS_SH_C2A * y; dY[4][1] = GS_SH_C2A * x; dY[4][2] = 0.0;
  dY[5][0] = 0.0; dY[5][1] = -GS_SH_C2A * z; dY[5][2] = -GS_SH_C2A * y;
  dY[6][0] = -2.0 * GS_SH_C2B * x; dY[6][1] = -2.0 * GS_SH_C2B * y; dY[6][2] = 4.0 * GS_SH_C2B * z;
  dY[7][0] = -GS_SH_C2A * z; dY[7][1] = 0.0; dY[7][2] = -GS_SH_C2A * x;
  dY[8][0] = 2.0 * GS_SH_C2C * x; dY[8][1] = -2.0 * GS_SH_C2C * y; dY[8][2] = 0.0;
  if (deg < 3) return;
  dY[9][0] = -6.0 * GS_SH_C3A * x * y; dY[9][1] = -3.0 * GS_SH_C3A * (xx - yy); dY[9][2] = 0.0;
  dY[10][0] = GS_SH_C3B * y * z; dY[10][1] = GS_SH_C3B * x * z; dY[10][2] = GS_SH_C3B * x * y;
  dY[11][0] = 2.0 * GS_SH_C3C * x * y; dY[11][1] = -GS_SH_C3C * (4.0 * zz - xx - 3.0 * yy);
  dY[11][2] = -8.0 * GS_SH_C3C * y * z;
  dY[12][0] = -6.0 * GS_SH_C3D * x * z; dY[12][1] = -6.0 * GS_SH_C3D * y * z;
  dY[12][2] = 3.0 * GS_SH_C3D * (2.0 * zz - xx - yy);
  dY[13][0] = -GS_SH_C3C * (4.0 * zz - 3.0 * xx - yy); dY[13][1] = 2.0 * GS_SH_C3C * x * y;
  dY[13][2] = -8.0 * GS_SH_C3C * x * z;
  dY[14][0] = 2.0 * GS_SH_C3E * x * z; dY[14][1] = -2.0 * GS_SH_C3E * y * z; dY[14][2] = GS_SH_C3E * (xx - yy);
  dY[15][0] = -3.0 * GS_SH_C3A * (xx - yy); dY[15][1] = 6.0 * GS_SH_C3A * x * y; dY[15][2] = 0.0;
}

}  // namespace gabsplat
