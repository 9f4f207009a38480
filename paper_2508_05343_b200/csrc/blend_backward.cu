// S4a / K7: the blend in reverse (gradients of sum_p <dL/dC(p), C(p)> with respect to the projected
// quantities of every primitive, including f2D and omega; PAPER.md:48, :129 -- derivation in DESIGN.md).
// Same CTA / pixel mapping as the forward kernel (blend_common.cuh): 64 threads per tile, 4 pixels per thread.
// Each warp replays the list of blended primitives the forward saved for its half tile, back to front, and
// recovers the transmittance in front of each primitive by division.  Per primitive a thread first sums the
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

constexpr int kReplay = 32;  // saved entries staged per warp and batch

// ABS: also accumulate sum |dL/dmu2D| per pixel (AbsGS densification statistic).
//
// Every warp replays, back to front, the list the forward saved for its half tile (BlendState): the
// primitives that were blended at one of the warp's 128 pixels, with the ballots of the blending lanes.  No
// tile list is walked, no skip / stop decision is re-taken, and the two warps of a CTA never synchronise.
// A lane recomputes G, cos, sin and alpha of its blended pixels with the forward's own functions (bit-identical
// alpha), recovers the transmittance in front of the primitive by division, and accumulates the gradient terms.
template <int K, bool ABS>
__global__ void __launch_bounds__(32, 16) blend_backward_kernel(Camera cam, const uint2* __restrict__ ranges,
                                                                       BlendState saved, const float4* __restrict__ packed,
                                                                       const float* __restrict__ final_T,
                                                                       const float* __restrict__ dL_dimage,
                                                                       float* __restrict__ grad2d) {
  pdl_wait();
  constexpr int R4 = packed_floats(K) / 4;
  constexpr int TL = K > 0 ? tail_floats(K) : 1;
  constexpr int NV = 9 + 3 * K + (ABS ? 2 : 0);
  constexpr int GF = grad2d_floats(K);
  // one warp per CTA: CTA b replays half tile order[b] (half tiles by descending saved-list length)
  __shared__ float4 s_rec1[kReplay * R4];
  __shared__ uint4 s_mask1[kReplay];
  __shared__ uint32_t s_id1[kReplay];
  const uint32_t half = __ldg(saved.order + blockIdx.x);
  const TileGeom g = tile_geom_at(cam, (int)(half >> 1), (int)(half & 1u), (int)threadIdx.x);
  const uint2 range = ranges[g.tile];
  const size_t HW = (size_t)cam.width * cam.height;
  const int cnt = (int)saved.counts[2 * g.tile + g.warp];
  const size_t base = 2 * (size_t)range.x + (size_t)g.warp * (range.y - range.x);
  float4* __restrict__ rec = s_rec1;

  float T[kSlots], gC[kSlots][3], B[kSlots][3];
#pragma unroll
  for (int s = 0; s < kSlots; ++s) {
    T[s] = 0.f;
    gC[s][0] = gC[s][1] = gC[s][2] = 0.f;
    if (g.inside[s]) {
      const size_t pix = (size_t)g.py[s] * cam.width + g.px;
      T[s] = final_T[pix];
      gC[s][0] = dL_dimage[pix]; gC[s][1] = dL_dimage[HW + pix]; gC[s][2] = dL_dimage[2 * HW + pix];
    }
    B[s][0] = cam.bg[0]; B[s][1] = cam.bg[1]; B[s][2] = cam.bg[2];  // colour behind the current primitive
  }

  constexpr int NL = reduce_left(NV);
  int my_idx[NL];
#pragma unroll
  for (int i = 0; i < NL; ++i) my_idx[i] = reduce_index<NV>(g.lane, i);

  // batches from the back: lane l of a batch stages saved entry end - 1 - l
  for (int end = cnt; end > 0; end -= kReplay) {
    const int m = min(kReplay, end);
    uint32_t my_id = 0;
    uint4 my_mask = make_uint4(0u, 0u, 0u, 0u);
    if (g.lane < m) {
      my_id = __ldg(saved.ids + base + (size_t)(end - 1 - g.lane));
      my_mask = __ldg(saved.masks + base + (size_t)(end - 1 - g.lane));
    }
    s_id1[g.lane] = my_id;
    s_mask1[g.lane] = my_mask;
#pragma unroll
    for (int it = 0; it < R4; ++it) {
      const int idx = it * 32 + g.lane;
      const int r = idx / R4, part = idx - r * R4;
      const uint32_t id_r = __shfl_sync(kFull, my_id, r);
      if (r < m) {
        float4 v = __ldg(packed + (size_t)id_r * R4 + part);
        if (part == 0) {  // mean relative to the tile origin, as the forward computes it: (hi - origin) + lo
          v.x = __fadd_rn(__fsub_rn(v.x, g.x0), v.z);
          v.y = __fadd_rn(__fsub_rn(v.y, g.y0), v.w);
        }
        rec[idx] = v;
      }
    }
    __syncwarp();
    for (int j = 0; j < m; ++j) {
      const uint4 mk = s_mask1[j];
      const float4 a = rec[j * R4], l = rec[j * R4 + 1], oc = rec[j * R4 + 2];
      const bool hit[kSlots] = {((mk.x >> g.lane) & 1u) != 0u, ((mk.y >> g.lane) & 1u) != 0u,
                                ((mk.z >> g.lane) & 1u) != 0u, ((mk.w >> g.lane) & 1u) != 0u};
      float tail[TL];
      if (K > 0) load_tail<K>(rec + j * R4, tail);
      const float dx = __fsub_rn(g.lx, a.x);
      const float ux = __fmul_rn(l.x, dx);
      ModulationEntry<K> me;
      modulation_entry<K>(tail, dx, me);
      float acc[NV];
#pragma unroll
      for (int i = 0; i < NV; ++i) acc[i] = 0.f;
      // sums over the thread's pixels of terms whose common factors (dx, L, 2 pi f2D) are applied once, below
      float Suu = 0.f, Suv = 0.f, Svv = 0.f, Squ = 0.f, Sqv = 0.f;
      float Sg[K > 0 ? K : 1], Sgy[K > 0 ? K : 1];
#pragma unroll
      for (int k = 0; k < K; ++k) Sg[k] = Sgy[k] = 0.f;
#pragma unroll
      for (int s = 0; s < kSlots; ++s) {
        if (!hit[s]) continue;
        float u, v;
        const float dy = __fsub_rn(g.ly[s], a.y);
        const float q = envelope_q(ux, l.y, l.z, dy, u, v);
        const float G = envelope_exp2(q);
        Modulation<K> e;
        modulation<K, true>(tail, me, dy, e);
        const float raw = __fmul_rn(__fmul_rn(oc.x, G), e.M);
        const float alpha = fminf(kAlphaMax, raw);
        const float om = 1.0f - alpha;
        const float Ti = __fdividef(T[s], om);  // transmittance in front of this primitive
        T[s] = Ti;
        const float aT = alpha * Ti;
        acc[6] += aT * gC[s][0]; acc[7] += aT * gC[s][1]; acc[8] += aT * gC[s][2];
        const float d0 = oc.y - B[s][0], d1 = oc.z - B[s][1], d2 = oc.w - B[s][2];  // colour minus what is behind
        const float galpha = Ti * (gC[s][0] * d0 + gC[s][1] * d1 + gC[s][2] * d2);
        B[s][0] = fmaf(alpha, d0, B[s][0]);  // = alpha c + (1 - alpha) B
        B[s][1] = fmaf(alpha, d1, B[s][1]);
        B[s][2] = fmaf(alpha, d2, B[s][2]);
        if (!(raw > kAlphaMax)) {  // the clamp min(0.99, .) has zero derivative when active
          const float gG = galpha * G;
          acc[5] += gG * e.M;
          const float ngM = -(gG * oc.x);   // -dL/dM
          const float gq = galpha * raw;    // dL/d(ln G)
          // the conic's gradient is accumulated in the whitened coordinates (u, v) of the envelope,
          // S = sum gq w w^T: its entries are O(gq) whatever the anisotropy of the footprint, where the sums of
          // gq dx^2, gq dx dy, gq dy^2 lose the thin direction of a needle that spans the screen in the other
          const float gqu = gq * u, gqv = gq * v;
          Suu += gqu * u; Suv += gqu * v; Svv += gqv * v;
          Squ += gqu; Sqv += gqv;
          float pdx = 0.f, pdy = 0.f;       // per-pixel d/d(dx), d/d(dy) through the phases (AbsGS only)
#pragma unroll
          for (int k = 0; k < K; ++k) {
            acc[9 + 2 * K + k] -= ngM * (e.cs[k] - 1.0f);
            const float gph = ngM * tail[2 * K + k] * e.sn[k];  // dL/d(phase in radians)
            Sg[k] += gph;
            Sgy[k] += gph * dy;
            if (ABS) { pdx += gph * tail[2 * k]; pdy += gph * tail[2 * k + 1]; }
          }
          if (ABS) {
            // G = 2^q, q = -(u^2 + v^2), u = L11 dx + L21 dy, v = L22 dy:  dL/dq = gq ln 2
            acc[9 + 3 * K] += fabsf(pdx + gq * (-1.3862943611198906f * u * l.x));
            acc[10 + 3 * K] += fabsf(pdy + gq * (-1.3862943611198906f * (u * l.y + v * l.z)));
          }
        }
      }
      {
        // conic, in whitened form: S = sum dL/d(ln G) w w^T  (the projection backward maps it to dL/dU)
        acc[2] = Suu;
        acc[3] = Suv;
        acc[4] = Svv;
        // mean: d = p - mu2D, so dL/dmu2D = -dL/dd;  dL/dd = dL/dq ln 2 (-2 u L11, -2 (u L21 + v L22)) + sum_k gph_k 2 pi f2D_k
        float gdx = -1.3862943611198906f * l.x * Squ;
        float gdy = -1.3862943611198906f * (l.y * Squ + l.z * Sqv);
#pragma unroll
        for (int k = 0; k < K; ++k) {
          gdx += Sg[k] * tail[2 * k];
          gdy += Sg[k] * tail[2 * k + 1];
          acc[9 + 2 * k] = Sg[k] * dx;
          acc[9 + 2 * k + 1] = Sgy[k];
        }
        acc[0] = -gdx; acc[1] = -gdy;
      }
      Butterfly<NV, 16>::run(acc, g.lane);
      float* dst = grad2d + (size_t)s_id1[j] * GF;
#pragma unroll
      for (int i = 0; i < NL; ++i)
        if (my_idx[i] >= 0 && acc[i] != 0.f) atomicAdd(dst + my_idx[i], acc[i]);
    }
    __syncwarp();
  }
}

template <int K, bool ABS>
cudaError_t launch_k(const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                     const gabsplat_fwd_out& fwd, const BlendState& saved, const float* dL, float* grad2d, cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  launch_pdl(blend_backward_kernel<K, ABS>, 2 * ntiles, 32, 0, st, cam, reinterpret_cast<const uint2*>(bin.tile_ranges), saved,
             reinterpret_cast<const float4*>(proj.packed), (const float*)fwd.final_T, dL, grad2d);
  launched();
  return cudaGetLastError();
}

template <bool ABS>
cudaError_t dispatch(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                     const gabsplat_fwd_out& fwd, const BlendState& saved, const float* dL, float* grad2d, cudaStream_t st) {
  switch (K) {
    case 0: return launch_k<0, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 1: return launch_k<1, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 2: return launch_k<2, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 3: return launch_k<3, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 4: return launch_k<4, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 5: return launch_k<5, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 6: return launch_k<6, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 7: return launch_k<7, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
    case 8: return launch_k<8, ABS>(cam, proj, bin, fwd, saved, dL, grad2d, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_blend_backward(int N, int K, bool want_abs, const Camera& cam, const gabsplat_projected& proj,
                                  const gabsplat_binning& bin, const gabsplat_fwd_out& fwd, const BlendState& saved,
                                  const float* dL_dimage, float* grad2d, cudaStream_t st) {
  // grad2d is all zero on entry: the caller zeroes the workspace once, the projection backward clears the rows it read
  (void)N;
  // launch order: half-tile pairs with the longest saved lists first
  const cudaError_t eo = launch_half_tile_order(saved.counts, 2 * cam.tiles_x * cam.tiles_y, saved.order, st);
  if (eo != cudaSuccess) return eo;
  return want_abs ? dispatch<true>(K, cam, proj, bin, fwd, saved, dL_dimage, grad2d, st)
                  : dispatch<false>(K, cam, proj, bin, fwd, saved, dL_dimage, grad2d, st);
}

}  // namespace gabsplat
