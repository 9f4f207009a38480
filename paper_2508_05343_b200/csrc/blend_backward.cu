// S4a / K7: the blend in reverse (gradients of sum_p <dL/dC(p), C(p)> with respect to the projected
// quantities of every primitive, including f2D and omega; PAPER.md:48, :129 -- derivation in DESIGN.md).
// Same CTA / pixel mapping and staging as the forward kernel (blend_common.cuh): 64 threads per tile, 4 pixels
// per thread.  Pixels walk the tile list back to front from the tile's deepest contributor and recover the
// transmittance in front of each primitive by division.  Per staged primitive a thread first sums the
// gradient contributions of its 4 pixels in registers; the 9+3K (+2) sums are then reduced over the warp with a
// butterfly that halves the number of live values at every exchange (one shuffle per value pair instead of
// five per value) and leaves value i on lane idx(i), so the warp issues ONE vector of atomic adds per primitive.
#include "blend_common.cuh"

namespace gabsplat {
namespace {

// ---- multi-value warp reduction ---------------------------------------------------------------------
// v[0..n) on every lane.  Exchange distance D: lanes with bit D clear keep values [0,H), the others keep
// [H,n) (H = ceil(n/2)); each sends the half it does not keep.  After distances 16,8,4,2,1 v[0] holds the warp
// total of value reduce_index(lane) (or padding).
template <int n, int D>
struct Butterfly {
  template <int N>
  static __device__ __forceinline__ void run(float (&v)[N], int lane) {
    constexpr int H = (n + 1) / 2;
    const bool upper = (lane & D) != 0;
#pragma unroll
    for (int i = 0; i < H; ++i) {
      const float lo = v[i];
      const float hi = (i + H < n) ? v[i + H] : 0.f;
      const float send = upper ? lo : hi;
      const float keep = upper ? hi : lo;
      v[i] = keep + __shfl_xor_sync(kFull, send, D);
    }
    Butterfly<H, D / 2>::run(v, lane);
  }
};
template <int n>
struct Butterfly<n, 0> {
  template <int N>
  static __device__ __forceinline__ void run(float (&)[N], int) {}
};

// Number of values left on every lane after the five exchanges (1 for N <= 32).
__host__ __device__ constexpr int reduce_left(int N) {
  for (int L = 0; L < 5; ++L) N = (N + 1) / 2;
  return N;
}

// Which of the N values lane `lane` holds in v[i] after Butterfly<N,16>; -1 if it holds padding.
template <int N>
__device__ __forceinline__ int reduce_index(int lane, int i) {
  int cnt[5];
  int n = N;
#pragma unroll
  for (int L = 0; L < 5; ++L) { cnt[L] = n; n = (n + 1) / 2; }
  int rel = i;
  bool valid = true;
#pragma unroll
  for (int L = 4; L >= 0; --L) {
    if (lane & (16 >> L)) rel += (cnt[L] + 1) / 2;
    valid = valid && rel < cnt[L];
  }
  return valid ? rel : -1;
}

// ABS: also accumulate sum |dL/dmu2D| per pixel (AbsGS densification statistic).
template <int K, bool ABS>
__global__ void __launch_bounds__(kBlendThreads) blend_backward_kernel(Camera cam, const uint2* __restrict__ ranges,
                                                                       const uint32_t* __restrict__ ids,
                                                                       const float4* __restrict__ packed,
                                                                       const float* __restrict__ final_T,
                                                                       const uint32_t* __restrict__ n_contrib,
                                                                       const float* __restrict__ dL_dimage,
                                                                       float* __restrict__ grad2d) {
  constexpr int R4 = packed_floats(K) / 4;
  constexpr int TL = K > 0 ? tail_floats(K) : 1;
  constexpr int NV = 9 + 3 * K + (ABS ? 2 : 0);
  constexpr int GF = grad2d_floats(K);
  __shared__ float4 s_rec[kBatch * R4];
  __shared__ uint32_t s_cnt[8];
  __shared__ uint32_t s_max[kBlendThreads / 32];
  const TileGeom g = tile_geom(cam);
  const uint2 range = ranges[g.tile];
  const size_t HW = (size_t)cam.width * cam.height;

  float T[kSlots], gC[kSlots][3], B[kSlots][3];
  uint32_t last[kSlots];
  uint32_t mx = 0;
#pragma unroll
  for (int s = 0; s < kSlots; ++s) {
    T[s] = 0.f; last[s] = 0;
    gC[s][0] = gC[s][1] = gC[s][2] = 0.f;
    if (g.inside[s]) {
      const size_t pix = (size_t)g.py[s] * cam.width + g.px;
      T[s] = final_T[pix];
      last[s] = n_contrib[pix];
      gC[s][0] = dL_dimage[pix]; gC[s][1] = dL_dimage[HW + pix]; gC[s][2] = dL_dimage[2 * HW + pix];
    }
    B[s][0] = cam.bg[0]; B[s][1] = cam.bg[1]; B[s][2] = cam.bg[2];  // colour behind the current primitive
    mx = max(mx, last[s]);
  }
  // the tile's deepest contributor
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) mx = max(mx, __shfl_xor_sync(kFull, mx, d));
  if (g.lane == 0) s_max[g.warp] = mx;
  __syncthreads();
  uint32_t n_eff = 0;
#pragma unroll
  for (int w = 0; w < kBlendThreads / 32; ++w) n_eff = max(n_eff, s_max[w]);

  constexpr int NL = reduce_left(NV);
  int my_idx[NL];
#pragma unroll
  for (int i = 0; i < NL; ++i) my_idx[i] = reduce_index<NV>(g.lane, i);

  // batches from the back: candidate c of a batch is 1-based list position end - c
  for (int end = (int)n_eff; end > 0; end -= kBatch) {
    const int m = min(kBatch, end);
    const int ns = stage_batch<K, true>(g, ids, packed, range.x, end - 1, m, s_rec, s_cnt);
    for (int j = 0; j < ns; ++j) {
      const float4 h0 = s_rec[j * R4], h1 = s_rec[j * R4 + 1];
      const uint32_t pos = __float_as_uint(h1.z);
      const float dx = __fsub_rn(g.lx, h0.x);
      const float ux = __fmul_rn(h0.z, dx);
      float dy[kSlots], q[kSlots], u[kSlots], v[kSlots];
      bool pass[kSlots];
      bool any = false;
#pragma unroll
      for (int s = 0; s < kSlots; ++s) {
        dy[s] = __fsub_rn(g.ly[s], h0.y);
        q[s] = envelope_q(ux, h0.w, h1.x, dy[s], u[s], v[s]);
        pass[s] = pos <= last[s] && !(q[s] < h1.y);
        any = any || pass[s];
      }
      if (!__any_sync(kFull, any)) continue;  // warp-uniform

      const float4 oc = s_rec[j * R4 + 2];
      float tail[TL];
      if (K > 0) load_tail<K>(s_rec + j * R4, tail);
      float acc[NV];
#pragma unroll
      for (int i = 0; i < NV; ++i) acc[i] = 0.f;
      bool hit_any = false;
#pragma unroll
      for (int s = 0; s < kSlots; ++s) {
        if (!pass[s]) continue;
        const float G = __expf(q[s]);
        Modulation<K> e;
        modulation<K, true>(tail, dx, dy[s], e);
        const float raw = __fmul_rn(__fmul_rn(oc.x, G), e.M);
        const float alpha = fminf(kAlphaMax, raw);
        if (alpha < kAlphaMin) continue;
        hit_any = true;
        const float om = 1.0f - alpha;
        const float Ti = __fdividef(T[s], om);  // transmittance in front of this primitive
        T[s] = Ti;
        const float aT = alpha * Ti;
        acc[6] += aT * gC[s][0]; acc[7] += aT * gC[s][1]; acc[8] += aT * gC[s][2];
        const float galpha = Ti * (gC[s][0] * (oc.y - B[s][0]) + gC[s][1] * (oc.z - B[s][1]) + gC[s][2] * (oc.w - B[s][2]));
        B[s][0] = alpha * oc.y + om * B[s][0];
        B[s][1] = alpha * oc.z + om * B[s][1];
        B[s][2] = alpha * oc.w + om * B[s][2];
        if (!(raw > kAlphaMax)) {  // the clamp min(0.99, .) has zero derivative when active
          acc[5] += galpha * G * e.M;
          const float gM = galpha * oc.x * G;
          const float gq = galpha * raw;  // dL/dq = g_G * G
          // q = -(u^2 + v^2), u = L11 dx + L21 dy, v = L22 dy
          float gdx = gq * (-2.0f * u[s] * h0.z);
          float gdy = gq * (-2.0f * (u[s] * h0.w + v[s] * h1.x));
          acc[2] += gq * (-0.5f * dx * dx);
          acc[3] += gq * (-dx * dy[s]);
          acc[4] += gq * (-0.5f * dy[s] * dy[s]);
#pragma unroll
          for (int k = 0; k < K; ++k) {
            acc[9 + 2 * K + k] += gM * (e.cs[k] - 1.0f);
            const float gph = -gM * tail[2 * K + k] * e.sn[k];  // dL/d(phase in radians)
            acc[9 + 2 * k] += gph * dx;
            acc[9 + 2 * k + 1] += gph * dy[s];
            gdx += gph * tail[2 * k];
            gdy += gph * tail[2 * k + 1];
          }
          acc[0] -= gdx; acc[1] -= gdy;
          if (ABS) { acc[9 + 3 * K] += fabsf(gdx); acc[10 + 3 * K] += fabsf(gdy); }
        }
      }
      if (!__any_sync(kFull, hit_any)) continue;
      Butterfly<NV, 16>::run(acc, g.lane);
      float* dst = grad2d + (size_t)__float_as_uint(h1.w) * GF;
#pragma unroll
      for (int i = 0; i < NL; ++i)
        if (my_idx[i] >= 0 && acc[i] != 0.f) atomicAdd(dst + my_idx[i], acc[i]);
    }
  }
}

template <int K, bool ABS>
cudaError_t launch_k(const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                     const gabsplat_fwd_out& fwd, const float* dL, float* grad2d, cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  blend_backward_kernel<K, ABS><<<ntiles, kBlendThreads, 0, st>>>(
      cam, reinterpret_cast<const uint2*>(bin.tile_ranges), bin.ids, reinterpret_cast<const float4*>(proj.packed),
      fwd.final_T, fwd.n_contrib, dL, grad2d);
  launched();
  return cudaGetLastError();
}

template <bool ABS>
cudaError_t dispatch(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                     const gabsplat_fwd_out& fwd, const float* dL, float* grad2d, cudaStream_t st) {
  switch (K) {
    case 0: return launch_k<0, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 1: return launch_k<1, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 2: return launch_k<2, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 3: return launch_k<3, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 4: return launch_k<4, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 5: return launch_k<5, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 6: return launch_k<6, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 7: return launch_k<7, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
    case 8: return launch_k<8, ABS>(cam, proj, bin, fwd, dL, grad2d, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_blend_backward(int N, int K, bool want_abs, const Camera& cam, const gabsplat_projected& proj,
                                  const gabsplat_binning& bin, const gabsplat_fwd_out& fwd, const float* dL_dimage,
                                  float* grad2d, cudaStream_t st) {
  cudaMemsetAsync(grad2d, 0, (size_t)N * grad2d_floats(K) * sizeof(float), st);
  return want_abs ? dispatch<true>(K, cam, proj, bin, fwd, dL_dimage, grad2d, st)
                  : dispatch<false>(K, cam, proj, bin, fwd, dL_dimage, grad2d, st);
}

}  // namespace gabsplat
