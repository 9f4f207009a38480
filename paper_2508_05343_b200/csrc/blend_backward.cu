// S4a / K7: the blend in reverse (gradients of sum_p <dL/dC(p), C(p)> with respect to the projected
// quantities of every primitive, including f2D and omega; PAPER.md:48, :129 -- derivation in DESIGN.md).
// One CTA per tile; pixels walk the tile list back to front from the tile's last contributor, recover the
// transmittance in front of each primitive, and the per-primitive sums over the tile's pixels are reduced
// across the warp before one atomic per value.
#include "blend_common.cuh"

namespace gabsplat {
namespace {

constexpr int kBlock = 256;

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  return v;
}

template <int K>
__global__ void __launch_bounds__(kBlock) blend_backward_kernel(Camera cam, const uint2* __restrict__ ranges,
                                                               const uint32_t* __restrict__ ids,
                                                               const float4* __restrict__ packed,
                                                               const float* __restrict__ final_T,
                                                               const uint32_t* __restrict__ n_contrib,
                                                               const float* __restrict__ dL_dimage, float* __restrict__ grad2d) {
  constexpr int R = packed_floats(K);
  constexpr int R4 = R / 4;
  constexpr int wo = weight_offset(K);
  __shared__ uint32_t s_ids[kBlock];
  __shared__ float4 s_rec[kBlock * R4];
  __shared__ uint32_t s_max[kBlock / 32];
  const int tid = threadIdx.x, lane = tid & 31;
  const int tile = blockIdx.x;
  const int tx = tile % cam.tiles_x, ty = tile / cam.tiles_x;
  const int lxi = tid & 15, lyi = tid >> 4;
  const int px = tx * kTile + lxi, py = ty * kTile + lyi;
  const bool inside = px < cam.width && py < cam.height;
  const float lx = (float)lxi, ly = (float)lyi;
  const float x0 = (float)(tx * kTile), y0 = (float)(ty * kTile);
  const uint2 range = ranges[tile];
  const size_t HW = (size_t)cam.width * cam.height, pix = (size_t)py * cam.width + px;

  float T = 0.f, gCr = 0.f, gCg = 0.f, gCb = 0.f;
  uint32_t last = 0;
  if (inside) {
    T = final_T[pix];
    last = n_contrib[pix];
    gCr = dL_dimage[pix]; gCg = dL_dimage[HW + pix]; gCb = dL_dimage[2 * HW + pix];
  }
  float Br = cam.bg[0], Bg = cam.bg[1], Bb = cam.bg[2];  // colour behind the current primitive
  // the tile's deepest contributor
  uint32_t mx = last;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
  if (lane == 0) s_max[tid >> 5] = mx;
  __syncthreads();
  uint32_t n_eff = 0;
#pragma unroll
  for (int w = 0; w < kBlock / 32; ++w) n_eff = max(n_eff, s_max[w]);

  // batches from the back: batch covers list positions (end - m, end], staged so that s_rec[j] is position end - j
  for (int end = (int)n_eff; end > 0; end -= kBlock) {
    const int m = min(kBlock, end);
    __syncthreads();
    if (tid < m) s_ids[tid] = ids[range.x + (uint32_t)(end - 1 - tid)];
    __syncthreads();
    for (int c = tid; c < m * R4; c += kBlock) {
      const int rec = c / R4, ch = c - rec * R4;
      float4 v = __ldg(packed + (size_t)s_ids[rec] * R4 + ch);
      if (ch == 0) {
        v.x = __fadd_rn(__fsub_rn(v.x, x0), v.z);
        v.y = __fadd_rn(__fsub_rn(v.y, y0), v.w);
      }
      s_rec[c] = v;
    }
    __syncthreads();
    for (int j = 0; j < m; ++j) {
      const uint32_t pos = (uint32_t)(end - j);  // 1-based position in the tile list
      const float* rec = reinterpret_cast<const float*>(s_rec + j * R4);
      const float4 a = s_rec[j * R4], l = s_rec[j * R4 + 1];
      PairEval<K> e;
      e.dx = __fsub_rn(lx, a.x);
      e.dy = __fsub_rn(ly, a.y);
      bool hit = pos <= last;
      float4 oc = make_float4(0.f, 0.f, 0.f, 0.f);
      if (hit) {
        const float q = envelope_q(l.x, l.y, l.z, e.dx, e.dy, e.u, e.v);
        hit = !(q < l.w);
        if (hit) {
          oc = s_rec[j * R4 + 2];
          e.G = __expf(q);
          modulation<K, true>(rec, e);
          e.raw = __fmul_rn(__fmul_rn(oc.x, e.G), e.M);
          e.alpha = fminf(kAlphaMax, e.raw);
          hit = !(e.alpha < kAlphaMin);
        }
      }
      if (!__any_sync(0xffffffffu, hit)) continue;
      float g[R];
#pragma unroll
      for (int v = 0; v < R; ++v) g[v] = 0.f;
      if (hit) {
        const float Ti = T / (1.0f - e.alpha);  // transmittance in front of this primitive
        T = Ti;
        const float aT = e.alpha * Ti;
        g[6] = aT * gCr; g[7] = aT * gCg; g[8] = aT * gCb;
        const float galpha = Ti * (gCr * (oc.y - Br) + gCg * (oc.z - Bg) + gCb * (oc.w - Bb));
        const float om = 1.0f - e.alpha;
        Br = e.alpha * oc.y + om * Br;
        Bg = e.alpha * oc.z + om * Bg;
        Bb = e.alpha * oc.w + om * Bb;
        if (!(e.raw > kAlphaMax)) {  // the clamp min(0.99, .) has zero derivative when active
          g[5] = galpha * e.G * e.M;
          const float gM = galpha * oc.x * e.G;
          const float gq = galpha * e.raw;  // dL/dq = g_G * G
          // q = -(u^2 + v^2), u = L11 dx + L21 dy, v = L22 dy
          float gdx = gq * (-2.0f * e.u * l.x);
          float gdy = gq * (-2.0f * (e.u * l.y + e.v * l.z));
          g[2] = gq * (-0.5f * e.dx * e.dx);
          g[3] = gq * (-e.dx * e.dy);
          g[4] = gq * (-0.5f * e.dy * e.dy);
#pragma unroll
          for (int k = 0; k < K; ++k) {
            g[wo + k] = gM * (e.cs[k] - 1.0f);
            const float gph = -gM * rec[wo + k] * e.sn[k] * kTwoPi;  // dL/d(phase in cycles)
            g[12 + 2 * k] = gph * e.dx;
            g[12 + 2 * k + 1] = gph * e.dy;
            gdx += gph * rec[12 + 2 * k];
            gdy += gph * rec[12 + 2 * k + 1];
          }
          g[0] = -gdx; g[1] = -gdy;
          g[9] = fabsf(gdx); g[10] = fabsf(gdy);
        }
      }
      float* dst = grad2d + (size_t)s_ids[j] * R;
#pragma unroll
      for (int v = 0; v < R; ++v) {
        if (v == 11 || (v >= 12 + 2 * K && v < wo) || v >= wo + K) continue;  // padding
        const float s = warp_sum(g[v]);
        if (lane == 0 && s != 0.f) atomicAdd(dst + v, s);
      }
    }
  }
}

template <int K>
cudaError_t launch_k(const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                     const gabsplat_fwd_out& fwd, const float* dL, float* grad2d, cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  blend_backward_kernel<K><<<ntiles, kBlock, 0, st>>>(cam, reinterpret_cast<const uint2*>(bin.tile_ranges), bin.ids,
                                                       reinterpret_cast<const float4*>(proj.packed), fwd.final_T,
                                                       fwd.n_contrib, dL, grad2d);
  launched();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_blend_backward(int N, int K, const Camera& cam, const gabsplat_projected& proj,
                                  const gabsplat_binning& bin, const gabsplat_fwd_out& fwd, const float* dL_dimage,
                                  float* grad2d, cudaStream_t st) {
  cudaMemsetAsync(grad2d, 0, (size_t)N * grad2d_floats(K) * sizeof(float), st);
  switch (K) {
    case 0: return launch_k<0>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 1: return launch_k<1>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 2: return launch_k<2>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 3: return launch_k<3>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 4: return launch_k<4>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 5: return launch_k<5>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 6: return launch_k<6>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 7: return launch_k<7>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
    case 8: return launch_k<8>(cam, proj, bin, fwd, dL_dimage, grad2d, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace gabsplat
