// S3 / K6: per-tile front-to-back blend of 2D Gabor primitives (PAPER.md:158 Eq.12, :162 Eq.13).
// One CTA per 16x16 tile, one pixel per thread; the tile's sorted list is staged through shared memory in
// batches of 256 packed records (sector-granular cooperative gather); the CTA stops when every pixel's
// transmittance is saturated.
#include "blend_common.cuh"

namespace gabsplat {
namespace {

constexpr int kBlock = 256;

// COUNT = the instrumented variant behind gabsplat_count_pairs: same decisions, and per pixel the number of
// list entries examined / past the envelope test / blended is written to `counters` instead of the image.
template <int K, bool COUNT>
__global__ void __launch_bounds__(kBlock) blend_forward_kernel(Camera cam, const uint2* __restrict__ ranges,
                                                              const uint32_t* __restrict__ ids,
                                                              const float4* __restrict__ packed, float* __restrict__ image,
                                                              float* __restrict__ final_T, uint32_t* __restrict__ n_contrib,
                                                              uint32_t* __restrict__ counters) {
  constexpr int R = packed_floats(K);
  constexpr int R4 = R / 4;
  __shared__ uint32_t s_ids[kBlock];
  __shared__ float4 s_rec[kBlock * R4];
  const int tid = threadIdx.x;
  const int tile = blockIdx.x;
  const int tx = tile % cam.tiles_x, ty = tile / cam.tiles_x;
  const int lxi = tid & 15, lyi = tid >> 4;
  const int px = tx * kTile + lxi, py = ty * kTile + lyi;
  const bool inside = px < cam.width && py < cam.height;
  const float lx = (float)lxi, ly = (float)lyi;
  const float x0 = (float)(tx * kTile), y0 = (float)(ty * kTile);
  const uint2 range = ranges[tile];
  const int n = (int)(range.y - range.x);

  float T = 1.0f, Cr = 0.f, Cg = 0.f, Cb = 0.f;
  uint32_t last = 0;
  uint32_t n_exam = 0, n_env = 0, n_blend = 0, n_env_last = 0;
  bool done = !inside;
  for (int b0 = 0; b0 < n; b0 += kBlock) {
    if (__syncthreads_and(done)) break;
    const int m = min(kBlock, n - b0);
    if (tid < m) s_ids[tid] = ids[range.x + b0 + tid];
    __syncthreads();
    for (int c = tid; c < m * R4; c += kBlock) {
      const int rec = c / R4, ch = c - rec * R4;
      float4 v = __ldg(packed + (size_t)s_ids[rec] * R4 + ch);
      if (ch == 0) {  // mean relative to the tile origin: (hi - origin) + lo
        v.x = __fadd_rn(__fsub_rn(v.x, x0), v.z);
        v.y = __fadd_rn(__fsub_rn(v.y, y0), v.w);
      }
      s_rec[c] = v;
    }
    __syncthreads();
    if (!done) {
      for (int j = 0; j < m; ++j) {
        const float* rec = reinterpret_cast<const float*>(s_rec + j * R4);
        const float4 a = s_rec[j * R4], l = s_rec[j * R4 + 1];
        PairEval<K> e;
        e.dx = __fsub_rn(lx, a.x);
        e.dy = __fsub_rn(ly, a.y);
        const float q = envelope_q(l.x, l.y, l.z, e.dx, e.dy, e.u, e.v);
        if (COUNT) ++n_exam;
        if (q < l.w) continue;  // envelope reject: o G < 1/255 and M <= 1
        if (COUNT) ++n_env;
        const float4 oc = s_rec[j * R4 + 2];
        e.G = __expf(q);
        modulation<K, false>(rec, e);
        e.raw = __fmul_rn(__fmul_rn(oc.x, e.G), e.M);
        e.alpha = fminf(kAlphaMax, e.raw);
        if (e.alpha < kAlphaMin) continue;
        const float Tn = __fmul_rn(T, __fsub_rn(1.0f, e.alpha));
        if (Tn < kTMin) { done = true; break; }
        const float wgt = __fmul_rn(e.alpha, T);
        Cr = __fmaf_rn(oc.y, wgt, Cr);
        Cg = __fmaf_rn(oc.z, wgt, Cg);
        Cb = __fmaf_rn(oc.w, wgt, Cb);
        T = Tn;
        last = (uint32_t)(b0 + j + 1);
        if (COUNT) { ++n_blend; n_env_last = n_env; }
      }
    }
  }
  if (COUNT) {
    if (inside) {
      reinterpret_cast<uint4*>(counters)[(size_t)py * cam.width + px] = make_uint4(n_exam, n_env, n_blend, n_env_last);
    }
    return;
  }
  if (inside) {
    const size_t HW = (size_t)cam.width * cam.height, pix = (size_t)py * cam.width + px;
    image[pix] = __fmaf_rn(T, cam.bg[0], Cr);
    image[HW + pix] = __fmaf_rn(T, cam.bg[1], Cg);
    image[2 * HW + pix] = __fmaf_rn(T, cam.bg[2], Cb);
    final_T[pix] = T;
    n_contrib[pix] = last;
  }
}

template <int K>
cudaError_t launch_k(const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                     const gabsplat_fwd_out& out, cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  blend_forward_kernel<K, false><<<ntiles, kBlock, 0, st>>>(cam, reinterpret_cast<const uint2*>(bin.tile_ranges), bin.ids,
                                                             reinterpret_cast<const float4*>(proj.packed), out.image,
                                                             out.final_T, out.n_contrib, nullptr);
  launched();
  return cudaGetLastError();
}

template <int K>
cudaError_t count_k(const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin, uint32_t* counters,
                    cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  blend_forward_kernel<K, true><<<ntiles, kBlock, 0, st>>>(cam, reinterpret_cast<const uint2*>(bin.tile_ranges), bin.ids,
                                                            reinterpret_cast<const float4*>(proj.packed), nullptr, nullptr,
                                                            nullptr, counters);
  launched();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_blend_forward(int K, const Camera& cam, const gabsplat_projected& proj,
                                 const gabsplat_binning& bin, const gabsplat_fwd_out& out, cudaStream_t st) {
  switch (K) {
    case 0: return launch_k<0>(cam, proj, bin, out, st);
    case 1: return launch_k<1>(cam, proj, bin, out, st);
    case 2: return launch_k<2>(cam, proj, bin, out, st);
    case 3: return launch_k<3>(cam, proj, bin, out, st);
    case 4: return launch_k<4>(cam, proj, bin, out, st);
    case 5: return launch_k<5>(cam, proj, bin, out, st);
    case 6: return launch_k<6>(cam, proj, bin, out, st);
    case 7: return launch_k<7>(cam, proj, bin, out, st);
    case 8: return launch_k<8>(cam, proj, bin, out, st);
  }
  return cudaErrorInvalidValue;
}

cudaError_t launch_count_pairs(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                               uint32_t* counters, cudaStream_t st) {
  switch (K) {
    case 0: return count_k<0>(cam, proj, bin, counters, st);
    case 1: return count_k<1>(cam, proj, bin, counters, st);
    case 2: return count_k<2>(cam, proj, bin, counters, st);
    case 3: return count_k<3>(cam, proj, bin, counters, st);
    case 4: return count_k<4>(cam, proj, bin, counters, st);
    case 5: return count_k<5>(cam, proj, bin, counters, st);
    case 6: return count_k<6>(cam, proj, bin, counters, st);
    case 7: return count_k<7>(cam, proj, bin, counters, st);
    case 8: return count_k<8>(cam, proj, bin, counters, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace gabsplat
