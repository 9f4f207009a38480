// S3 / K6: per-tile front-to-back blend of 2D Gabor primitives (PAPER.md:158 Eq.12, :162 Eq.13).
// One CTA of 64 threads per 16x16 tile, 4 pixels per thread; the tile's sorted list is staged through shared
// memory in batches with an exact tile-vs-ellipse pre-filter (blend_common.cuh); a staged record is read once
// per thread and evaluated at the thread's 4 pixels; the CTA stops when every pixel's transmittance is
// saturated (block-wide vote).
#include "blend_common.cuh"

namespace gabsplat {
namespace {

// COUNT = the instrumented variant behind gabsplat_count_pairs: same decisions; per pixel the number of list
// entries examined / past the envelope test / blended is written to `counters` instead of the image.
// SAVE = also record, per warp (half tile), the primitives blended at one of its pixels and the ballots of the
// blending lanes (common.cuh BlendState): the backward replays exactly this list.
#ifdef GS_FWD_STAGING_CPASYNC
// The staging experiment north_star (3) asks for ("TMA bulk copies where they pay"), kept buildable so that its
// measurement can be repeated (GABSPLAT_NVCC_FLAGS=-DGS_FWD_STAGING_CPASYNC python -m paper_2508_05343_b200.build --force):
// the batches of a tile's list staged by a three-deep software pipeline of asynchronous copies (cp.async / LDGSTS; the
// gathers are data-dependent 16-byte pieces of records, which the tensor form of TMA cannot address).  Measured at the
// headline config: 0.552 ms (64-entry batches, 10 CTAs/SM) and 0.579 ms (128-entry batches, 7 CTAs/SM by shared memory)
// against 0.527 ms for the synchronous staging below -- the loads it hides were already covered by the other CTAs of
// the SM, and it costs occupancy and a batch of filtering past the point where the tile saturates.  DESIGN.md 7.4.
// ---- asynchronous copies global -> shared (LDGSTS): the staging pipeline below keeps them in flight while a batch is blended
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

#ifndef GS_FWD_BATCH
#define GS_FWD_BATCH 64
#endif
constexpr int kFwdBatch = GS_FWD_BATCH;              // list entries filtered per batch
constexpr int kFwdPer = kFwdBatch / kBlendThreads;   // ... per thread
#endif

#ifndef GS_FWD_MINB
#define GS_FWD_MINB 10
#endif
template <int K, bool COUNT, bool SAVE>
__global__ void __launch_bounds__(kBlendThreads, GS_FWD_MINB) blend_forward_kernel(Camera cam, const uint32_t* __restrict__ order,
                                                                      const uint2* __restrict__ ranges,
                                                                      const uint32_t* __restrict__ ids,
                                                                      const float4* __restrict__ packed,
                                                                      const float4* __restrict__ colour,
                                                                      float* __restrict__ image, float* __restrict__ final_T,
                                                                      uint32_t* __restrict__ n_contrib,
                                                                      uint32_t* __restrict__ counters, BlendState save,
                                                                      uint32_t* __restrict__ tile_work) {
  pdl_wait();
  constexpr int R4 = packed_floats(K) / 4;
  constexpr int TL = K > 0 ? 4 * ((3 * K + 3) / 4) : 1;
#ifdef GS_FWD_STAGING_CPASYNC
  __shared__ float4 s_rec[2][kFwdBatch * R4];
  __shared__ float4 s_head[kFwdBatch * 2];
  __shared__ uint32_t s_ids[kFwdBatch];
  __shared__ uint32_t s_cnt[kFwdPer * (kBlendThreads / 32)];
#else
  __shared__ float4 s_rec[kBatch * R4];
  __shared__ uint32_t s_cnt[8];
#endif
  const TileGeom g = tile_geom(cam, order);
  const uint2 range = ranges[g.tile];
  const int n = (int)(range.y - range.x);

  float T[kSlots], Cr[kSlots], Cg[kSlots], Cb[kSlots];
  uint32_t last[kSlots];
  bool done[kSlots];
  uint32_t n_env[kSlots], n_blend[kSlots], n_env_last[kSlots], stop_pos[kSlots];
#pragma unroll
  for (int s = 0; s < kSlots; ++s) {
    T[s] = 1.0f; Cr[s] = Cg[s] = Cb[s] = 0.f;
    last[s] = 0;
    done[s] = !g.inside[s];
    n_env[s] = n_blend[s] = n_env_last[s] = 0;
    stop_pos[s] = 0;
  }

#ifdef GS_FWD_STAGING_CPASYNC
  const int tid = threadIdx.x;
  // ids of batch b -> registers
  auto load_ids = [&](int b, uint32_t (&idv)[kFwdPer]) {
#pragma unroll
    for (int r = 0; r < kFwdPer; ++r) {
      const int p = b * kFwdBatch + r * kBlendThreads + tid;
      idv[r] = p < n ? __ldg(ids + range.x + (uint32_t)p) : 0u;
    }
  };
  // heads of batch b -> s_head, asynchronously; every thread copies (and later filters) its own candidates
  auto issue_heads = [&](int b, const uint32_t (&idv)[kFwdPer]) {
#pragma unroll
    for (int r = 0; r < kFwdPer; ++r) {
      const int c = r * kBlendThreads + tid;
      if (b * kFwdBatch + c < n) {
        const float4* src = packed + (size_t)idv[r] * R4;
        cp_async16(&s_head[2 * c], src);
        cp_async16(&s_head[2 * c + 1], src + 1);
        s_ids[c] = idv[r];
      }
    }
  };
  // Filters batch b (its heads have landed in s_head), compacts the survivors in list order into s_rec[buf] -- heads by
  // plain stores, tails by asynchronous copies -- and returns their number.  Contains one __syncthreads.
  auto filter_compact = [&](int b, int buf) -> int {
    float4 h0[kFwdPer], h1[kFwdPer];
    uint32_t bal[kFwdPer];
    bool keep[kFwdPer];
#pragma unroll
    for (int r = 0; r < kFwdPer; ++r) {
      const int c = r * kBlendThreads + tid;
      const int p = b * kFwdBatch + c;
      keep[r] = false;
      if (p < n) {
        const float4 a = s_head[2 * c], l = s_head[2 * c + 1];
        // mean relative to the tile origin: (hi - origin) + lo
        const float mx = __fadd_rn(__fsub_rn(a.x, g.x0), a.z);
        const float my = __fadd_rn(__fsub_rn(a.y, g.y0), a.w);
        h0[r] = make_float4(mx, my, l.x, l.y);
        h1[r] = make_float4(l.z, l.w, __uint_as_float((uint32_t)p + 1u), __uint_as_float(s_ids[c]));
        keep[r] = tile_may_pass(mx, my, l.x, l.y, l.z, l.w);
      }
      bal[r] = __ballot_sync(kFull, keep[r]);
      if (g.lane == 0) s_cnt[r * (kBlendThreads / 32) + g.warp] = __popc(bal[r]);
    }
    __syncthreads();
    constexpr int kGroups = kFwdPer * (kBlendThreads / 32);
    uint32_t total = 0;
    uint32_t base[kFwdPer];
#pragma unroll
    for (int r = 0; r < kFwdPer; ++r) base[r] = 0;
#pragma unroll
    for (int q = 0; q < kGroups; ++q) {
#pragma unroll
      for (int r = 0; r < kFwdPer; ++r)
        if (q == r * (kBlendThreads / 32) + g.warp) base[r] = total;
      total += s_cnt[q];
    }
    const uint32_t lt = (1u << g.lane) - 1u;
#pragma unroll
    for (int r = 0; r < kFwdPer; ++r) {
      if (keep[r]) {
        const uint32_t slot = base[r] + __popc(bal[r] & lt);
        float4* dst = &s_rec[buf][slot * R4];
        dst[0] = h0[r];
        dst[1] = h1[r];
        const uint32_t pid = __float_as_uint(h1[r].w);
        const float4* src = packed + (size_t)pid * R4;
#pragma unroll
        for (int ch = 2; ch < R4; ++ch) cp_async16(dst + ch, (ch == 2 && colour) ? colour + pid : src + ch);
      }
    }
    return (int)total;
  };

#endif
  int walked = n;                                              // list entries consumed when the tile finished
  uint32_t n_saved = 0;                                        // warp-uniform
  const size_t save_at = 2 * (size_t)range.x + (size_t)g.warp * n;  // this warp's slice of save.ids / save.masks
  uint32_t* save_id = SAVE ? save.ids + save_at : nullptr;          // lane 0's write cursors
  uint4* save_mask = SAVE ? save.masks + save_at : nullptr;
#ifdef GS_FWD_STAGING_CPASYNC
  const int nbatch = (n + kFwdBatch - 1) / kFwdBatch;
  uint32_t idn[kFwdPer];   // ids of the batch whose heads are issued next
  int ns = 0;              // survivors of the batch about to be blended
  if (nbatch > 0) {        // prologue: the only exposed latencies of the tile
    load_ids(0, idn);
    issue_heads(0, idn);
    if (nbatch > 1) load_ids(1, idn);
    cp_async_wait_all();
    ns = filter_compact(0, 0);
    if (nbatch > 1) issue_heads(1, idn);
    if (nbatch > 2) load_ids(2, idn);
    cp_async_wait_all();
    __syncthreads();
  }
  for (int b = 0; b < nbatch; ++b) {
    const bool all_done = done[0] && done[1] && done[2] && done[3];
    if (__syncthreads_and(all_done)) { walked = b * kFwdBatch; break; }
    int ns_next = 0;
    if (b + 1 < nbatch) {
      ns_next = filter_compact(b + 1, (b + 1) & 1);
      if (b + 2 < nbatch) issue_heads(b + 2, idn);
      if (b + 3 < nbatch) load_ids(b + 3, idn);
    }
    const float4* __restrict__ recs = s_rec[b & 1];
    const int nj = __all_sync(kFull, all_done) ? 0 : ns;  // warp-uniform: the votes below need every lane
#define GS_FWD_RECS recs
#define GS_FWD_NJ nj
#else
  for (int b0 = 0; b0 < n; b0 += kBatch) {
    const bool all_done = done[0] && done[1] && done[2] && done[3];
    if (__syncthreads_and(all_done)) { walked = b0; break; }
    const int m = min(kBatch, n - b0);
    const int ns = stage_batch<K, false>(g, ids, packed, colour, range.x, b0, m, s_rec, s_cnt);
    if (__all_sync(kFull, all_done)) continue;  // warp-uniform: the votes below need every lane
#define GS_FWD_RECS s_rec
#define GS_FWD_NJ ns
#endif
    for (int j = 0; j < GS_FWD_NJ; ++j) {
      const float4 h0 = GS_FWD_RECS[j * R4], h1 = GS_FWD_RECS[j * R4 + 1];
      const float dx = __fsub_rn(g.lx, h0.x);
      const float ux = __fmul_rn(h0.z, dx);
      float dy[kSlots], q[kSlots];
      bool pass[kSlots];
      bool any = false;
#pragma unroll
      for (int s = 0; s < kSlots; ++s) {
        float u, v;
        dy[s] = __fsub_rn(g.ly[s], h0.y);
        q[s] = envelope_q(ux, h0.w, h1.x, dy[s], u, v);
        pass[s] = !(q[s] < h1.y) && !done[s];  // envelope reject: o G < 1/255 and M <= 1
        any = any || pass[s];
      }
      if (!__any_sync(kFull, any)) continue;  // warp-uniform
      const float4 oc = GS_FWD_RECS[j * R4 + 2];
      float tail[TL];
      if (K > 0) load_tail<K>(GS_FWD_RECS + j * R4, tail);
      const uint32_t pos = __float_as_uint(h1.z);
      ModulationEntry<K> me;
      modulation_entry<K>(tail, dx, me);
      // The four pixels of a thread are evaluated together, without branches (83 % of the slots of an evaluated
      // entry hold a passing lane anyway): four independent exp2 / cosine chains keep the pipes busy where one
      // chain per branch left the issue slots waiting on MUFU latency.  Lanes that failed the envelope test get
      // alpha = 0 by a select, never by arithmetic.
      float alpha[kSlots];
#pragma unroll
      for (int s = 0; s < kSlots; ++s) {
        if (COUNT && pass[s]) ++n_env[s];
        const float G = envelope_exp2(q[s]);
        Modulation<K> e;
        modulation<K, false>(tail, me, dy[s], e);
        const float raw = __fmul_rn(__fmul_rn(oc.x, G), e.M);
        alpha[s] = pass[s] ? fminf(kAlphaMax, raw) : 0.0f;
      }
#pragma unroll
      for (int s = 0; s < kSlots; ++s) {
        const bool hit = alpha[s] >= kAlphaMin;
        if (!__any_sync(kFull, hit)) continue;  // warp-uniform
        if (!hit) continue;
        const float Tn = __fmul_rn(T[s], __fsub_rn(1.0f, alpha[s]));
        if (Tn < kTMin) {
          done[s] = true;
          if (COUNT) stop_pos[s] = pos;
          continue;
        }
        const float wgt = __fmul_rn(alpha[s], T[s]);
        Cr[s] = __fmaf_rn(oc.y, wgt, Cr[s]);
        Cg[s] = __fmaf_rn(oc.z, wgt, Cg[s]);
        Cb[s] = __fmaf_rn(oc.w, wgt, Cb[s]);
        T[s] = Tn;
        last[s] = pos;
        if (COUNT) { ++n_blend[s]; n_env_last[s] = n_env[s]; }
      }
      if (SAVE) {
        // most evaluated entries blend at no pixel of the warp (M too small): one vote decides, the four ballots
        // and the two stores are paid only by entries that go to the list
        // (a pixel blended this entry iff its last-contributor position now is the entry's)
        const bool b0 = last[0] == pos, b1 = last[1] == pos, b2 = last[2] == pos, b3 = last[3] == pos;
        if (__any_sync(kFull, b0 || b1 || b2 || b3)) {
          uint4 m;
          m.x = __ballot_sync(kFull, b0); m.y = __ballot_sync(kFull, b1);
          m.z = __ballot_sync(kFull, b2); m.w = __ballot_sync(kFull, b3);
          if (g.lane == 0) {
            *save_id++ = __float_as_uint(h1.w);
            *save_mask++ = m;
          }
          ++n_saved;
        }
      }
    }
#ifdef GS_FWD_STAGING_CPASYNC
    cp_async_wait_all();   // tails of batch b + 1, heads of batch b + 2: they had the whole batch to land
    __syncthreads();
    ns = ns_next;
#endif
  }
  if (SAVE && g.lane == 0) save.counts[2 * g.tile + g.warp] = n_saved;
  if (tile_work && threadIdx.x == 0) tile_work[g.tile] = (uint32_t)walked;   // the launch-order hint of a later render
  const size_t HW = (size_t)cam.width * cam.height;
#pragma unroll
  for (int s = 0; s < kSlots; ++s) {
    if (!g.inside[s]) continue;
    const size_t pix = (size_t)g.py[s] * cam.width + g.px;
    if (COUNT) {
      // examined = list entries visited before the pixel stopped (the stopping entry included)
      const uint32_t n_exam = stop_pos[s] ? stop_pos[s] : (uint32_t)n;
      reinterpret_cast<uint4*>(counters)[pix] = make_uint4(n_exam, n_env[s], n_blend[s], n_env_last[s]);
    } else {
      image[pix] = __fmaf_rn(T[s], cam.bg[0], Cr[s]);
      image[HW + pix] = __fmaf_rn(T[s], cam.bg[1], Cg[s]);
      image[2 * HW + pix] = __fmaf_rn(T[s], cam.bg[2], Cb[s]);
      final_T[pix] = T[s];
      n_contrib[pix] = last[s];
    }
  }
}

template <int K, bool COUNT, bool SAVE>
cudaError_t launch_k(const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin, const float4* colour,
                     float* image, float* final_T, uint32_t* n_contrib, uint32_t* counters, const BlendState* save,
                     uint32_t* tile_work, cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  launch_pdl(blend_forward_kernel<K, COUNT, SAVE>, ntiles, kBlendThreads, 0, st, cam, (const uint32_t*)bin.tile_order,
             reinterpret_cast<const uint2*>(bin.tile_ranges), (const uint32_t*)bin.ids, reinterpret_cast<const float4*>(proj.packed),
             colour, image, final_T, n_contrib, counters, save ? *save : BlendState{nullptr, nullptr, nullptr, nullptr}, tile_work);
  launched();
  return cudaGetLastError();
}

template <bool COUNT, bool SAVE>
cudaError_t dispatch(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin, const float4* colour,
                     float* image, float* final_T, uint32_t* n_contrib, uint32_t* counters, const BlendState* save,
                     uint32_t* tile_work, cudaStream_t st) {
  switch (K) {
    case 0: return launch_k<0, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 1: return launch_k<1, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 2: return launch_k<2, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 3: return launch_k<3, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 4: return launch_k<4, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 5: return launch_k<5, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 6: return launch_k<6, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 7: return launch_k<7, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
    case 8: return launch_k<8, COUNT, SAVE>(cam, proj, bin, colour, image, final_T, n_contrib, counters, save, tile_work, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace

cudaError_t launch_blend_forward(int K, const Camera& cam, const gabsplat_projected& proj,
                                 const gabsplat_binning& bin, const gabsplat_fwd_out& out, const BlendState* save,
                                 cudaStream_t st) {
  return save ? dispatch<false, true>(K, cam, proj, bin, nullptr, out.image, out.final_T, out.n_contrib, nullptr, save, out.tile_work, st)
              : dispatch<false, false>(K, cam, proj, bin, nullptr, out.image, out.final_T, out.n_contrib, nullptr, nullptr, out.tile_work, st);
}

namespace {
// (opacity, sum_k omega_k |f2D_k|, depth, 1) per primitive: the "colours" of the auxiliary renders
__global__ void __launch_bounds__(256) aux_values_kernel(int N, int K, const uint32_t* __restrict__ tiles_touched,
                                                         const float* __restrict__ packed, const float* __restrict__ depth,
                                                         const float2* __restrict__ freq2d, const float* __restrict__ weights,
                                                         float4* __restrict__ aux) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
  if (tiles_touched[i] != 0) {
    float fm = 0.f;
    for (int k = 0; k < K; ++k) {
      const float2 f = freq2d[(size_t)i * K + k];
      fm = fmaf(weights[(size_t)i * K + k], sqrtf(f.x * f.x + f.y * f.y), fm);
    }
    v = make_float4(packed[(size_t)i * packed_floats(K) + 8], fm, depth[i], 1.0f);  // the opacity the blend uses (variants fold into it)
  }
  aux[i] = v;
}
}  // namespace

cudaError_t launch_blend_aux(int N, int K, const float* weights, const Camera& cam, const gabsplat_projected& proj,
                             const gabsplat_binning& bin, float4* aux, float* image, float* final_T, uint32_t* n_contrib,
                             cudaStream_t st) {
  if (N > 0) {
    aux_values_kernel<<<(N + 255) / 256, 256, 0, st>>>(N, K, proj.tiles_touched, proj.packed,
                                                       proj.depth, reinterpret_cast<const float2*>(proj.freq2d), weights, aux);
    launched();
  }
  Camera c = cam;
  c.bg[0] = c.bg[1] = c.bg[2] = 0.f;
  return dispatch<false, false>(K, c, proj, bin, aux, image, final_T, n_contrib, nullptr, nullptr, nullptr, st);
}

cudaError_t launch_count_pairs(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin,
                               uint32_t* counters, cudaStream_t st) {
  return dispatch<true, false>(K, cam, proj, bin, nullptr, nullptr, nullptr, nullptr, counters, nullptr, nullptr, st);
}

}  // namespace gabsplat

// ---- instrumentation: the forward's decisions at selected pixels ---------------------------------------
// gabsplat_trace_pixels: one thread per selected pixel walks its tile's list with the forward kernel's own functions
// (blend_common.cuh: same operands, same round-to-nearest operation sequence, so every alpha, every skip / stop
// decision and the accumulated colour are bit-identical to blend_forward_kernel's) and writes the 1-based list
// position of every entry it blends, bit 31 set when min(0.99, .) was active (what the backward reads as "zero
// derivative").  The parity tests hand these decisions to the oracle at the pixels whose decisions sit within
// fp32 error of a threshold (reading C18) and compare the trace's colour with the image bit for bit.
namespace gabsplat {
namespace {

template <int K>
__global__ void __launch_bounds__(128) trace_pixels_kernel(Camera cam, const uint2* __restrict__ ranges,
                                                           const uint32_t* __restrict__ ids, const float4* __restrict__ packed,
                                                           int n, const int2* __restrict__ pixels,
                                                           const uint32_t* __restrict__ offsets, uint32_t* __restrict__ entries,
                                                           float4* __restrict__ colour_T, uint4* __restrict__ info) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  constexpr int R4 = packed_floats(K) / 4;
  constexpr int TL = K > 0 ? tail_floats(K) : 1;
  const int2 p = pixels[i];
  if (p.x < 0 || p.y < 0 || p.x >= cam.width || p.y >= cam.height) {  // not a pixel of this image: flagged, nothing walked
    colour_T[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    info[i] = make_uint4(0u, 0u, 0u, 1u);
    return;
  }
  const int tx = p.x / kTile, ty = p.y / kTile;
  const uint2 range = ranges[ty * cam.tiles_x + tx];
  const float x0 = (float)(tx * kTile), y0 = (float)(ty * kTile);
  const float lx = (float)(p.x - tx * kTile), ly = (float)(p.y - ty * kTile);
  const uint32_t cap = offsets[i + 1] >= offsets[i] ? offsets[i + 1] - offsets[i] : 0u;  // descending offsets: no slice
  uint32_t* out = entries + offsets[i];
  float T = 1.0f, Cr = 0.f, Cg = 0.f, Cb = 0.f;
  uint32_t last = 0, stop = 0, nb = 0;
  for (uint32_t e = range.x; e < range.y; ++e) {
    const uint32_t id = ids[e];
    const float4* rec = packed + (size_t)id * R4;
    const float4 a = rec[0], l = rec[1], oc = rec[2];
    const float mx = __fadd_rn(__fsub_rn(a.x, x0), a.z), my = __fadd_rn(__fsub_rn(a.y, y0), a.w);
    const float dx = __fsub_rn(lx, mx), dy = __fsub_rn(ly, my);
    const float ux = __fmul_rn(l.x, dx);
    float u, v;
    const float q = envelope_q(ux, l.y, l.z, dy, u, v);
    if (q < l.w) continue;  // envelope reject
    float tail[TL];
    if (K > 0) load_tail<K>(rec, tail);
    ModulationEntry<K> me;
    modulation_entry<K>(tail, dx, me);
    Modulation<K> m;
    modulation<K, false>(tail, me, dy, m);
    const float raw = __fmul_rn(__fmul_rn(oc.x, envelope_exp2(q)), m.M);
    const float alpha = fminf(kAlphaMax, raw);
    if (!(alpha >= kAlphaMin)) continue;
    const uint32_t pos = e - range.x + 1u;
    const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
    if (Tn < kTMin) { stop = pos; break; }
    const float wgt = __fmul_rn(alpha, T);
    Cr = __fmaf_rn(oc.y, wgt, Cr);
    Cg = __fmaf_rn(oc.z, wgt, Cg);
    Cb = __fmaf_rn(oc.w, wgt, Cb);
    T = Tn;
    last = pos;
    if (nb < cap) out[nb] = pos | (raw > kAlphaMax ? 0x80000000u : 0u);
    ++nb;
  }
  colour_T[i] = make_float4(__fmaf_rn(T, cam.bg[0], Cr), __fmaf_rn(T, cam.bg[1], Cg), __fmaf_rn(T, cam.bg[2], Cb), T);
  info[i] = make_uint4(last, nb, stop, 0u);
}

}  // namespace

cudaError_t launch_trace_pixels(int K, const Camera& cam, const gabsplat_projected& proj, const gabsplat_binning& bin, int n,
                                const int32_t* pixels, const uint32_t* offsets, uint32_t* entries, float* colour_T,
                                uint32_t* info, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  const dim3 grid((n + 127) / 128), block(128);
#define GABSPLAT_TRACE(KK)                                                                                              \
  case KK:                                                                                                              \
    trace_pixels_kernel<KK><<<grid, block, 0, st>>>(cam, reinterpret_cast<const uint2*>(bin.tile_ranges), bin.ids,      \
                                                    reinterpret_cast<const float4*>(proj.packed), n,                    \
                                                    reinterpret_cast<const int2*>(pixels), offsets, entries,            \
                                                    reinterpret_cast<float4*>(colour_T), reinterpret_cast<uint4*>(info)); \
    break;
  switch (K) {
    GABSPLAT_TRACE(0) GABSPLAT_TRACE(1) GABSPLAT_TRACE(2) GABSPLAT_TRACE(3) GABSPLAT_TRACE(4)
    GABSPLAT_TRACE(5) GABSPLAT_TRACE(6) GABSPLAT_TRACE(7) GABSPLAT_TRACE(8)
    default: return cudaErrorInvalidValue;
  }
#undef GABSPLAT_TRACE
  launched();
  return cudaGetLastError();
}

// instrumentation: cos / sin of a raw radian phase exactly as modulation<> evaluates them (the MUFU path)
namespace {
__global__ void __launch_bounds__(256) probe_sincos_kernel(int n, const float* __restrict__ phase, float* __restrict__ c,
                                                           float* __restrict__ s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float tail[4] = {0.f, 1.0f, 1.0f, 0.f};  // K = 1: (2 pi f2D.x, 2 pi f2D.y, omega)
  ModulationEntry<1> me;
  modulation_entry<1>(tail, 0.f, me);
  Modulation<1> m;
  modulation<1, true>(tail, me, phase[i], m);  // phase = fma(1, phase, 0)
  c[i] = m.cs[0];
  s[i] = m.sn[0];
}
}  // namespace

cudaError_t launch_probe_sincos(int n, const float* phase, float* c, float* s, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  probe_sincos_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, phase, c, s);
  launched();
  return cudaGetLastError();
}

}  // namespace gabsplat
