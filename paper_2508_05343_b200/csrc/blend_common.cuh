// Shared by the forward and the backward blend kernels (S3 / S4a): the CTA / pixel mapping, the staging of a
// tile's sorted list through shared memory with an exact tile-vs-ellipse pre-filter, and the evaluation of one
// 2D Gabor primitive at one pixel (Eq.12).  Both kernels call the same functions, written with
// explicit round-to-nearest intrinsics (no compiler-chosen contraction), so that they take bit-identical
// skip / clamp decisions.
//
// Mapping.  A warp owns half a 16x16 tile (16x8 pixels) and every thread kSlots = 4 pixels: lane l of warp w
// owns column l & 15 and rows 8w + 2s + (l >> 4), s = 0..3.  Slot s of a warp is therefore a 16x2 strip.  The
// forward runs the two warps of a tile as one CTA (they share the staging); the backward, whose warps replay
// independent lists, runs every half tile as a CTA of its own.
// A staged record is read from shared memory once per thread and used for 4 pixels.
//
// Staging.  The tile's list is consumed in batches of kBatch entries.  Each thread fetches the 32-byte head of
// 2 entries (mean, Cholesky factor of the conic, envelope threshold) and tests whether ANY point of the tile's
// pixel rectangle can pass the per-pixel envelope test q >= qmin (minimum of the quadratic form over the
// rectangle, conservative by a relative margin).  Survivors are compacted in list order into shared memory
// (ballot + prefix over the 4 warp-rows), carrying their 1-based list position, and only their tails (colour,
// frequencies, weights) are gathered.  Entries that no pixel of the tile can see cost 32 bytes and ~30 flops
// instead of 256 pair evaluations.  The filter never changes a result: a culled entry fails the envelope test
// at every pixel of the tile.
#pragma once

#include "common.cuh"

namespace gabsplat {

constexpr int kBlendThreads = 64;
constexpr int kSlots = 4;
constexpr int kBatch = 128;
constexpr unsigned kFull = 0xffffffffu;

// shared-memory record of a surviving entry, floats (R = packed_floats(K), R4 = R / 4 float4):
//  [0..3]  mx, my (mean relative to the tile origin), L11, L21
//  [4..7]  L22, qmin, list position (1-based, uint bits), primitive id (uint bits)
//  [8..11] opacity, r, g, b
//  [12..]  2 pi f2D (x,y) * K, omega * K, padding    (verbatim tail of the packed record)

struct TileGeom {
  int tile, tx, ty, warp, lane, lxi;
  float lx;             // pixel column relative to the tile origin
  float ly[kSlots];     // pixel rows relative to the tile origin
  int px, py[kSlots];
  bool inside[kSlots];
  float x0, y0;         // tile origin in pixels
};

// CTA b works on tile order[b]: the tiles by descending work (binning.cu tile_order_kernel)
__device__ __forceinline__ TileGeom tile_geom_at(const Camera& cam, int tile, int warp, int lane);
__device__ __forceinline__ TileGeom tile_geom(const Camera& cam, const uint32_t* __restrict__ order) {
  return tile_geom_at(cam, (int)__ldg(order + blockIdx.x), threadIdx.x >> 5, threadIdx.x & 31);
}
// geometry of lane `lane` of half `warp` (rows 8 warp .. 8 warp + 7) of tile `tile`
__device__ __forceinline__ TileGeom tile_geom_at(const Camera& cam, int tile, int warp, int lane) {
  TileGeom g;
  g.tile = tile;
  g.tx = g.tile % cam.tiles_x;
  g.ty = g.tile / cam.tiles_x;
  g.warp = warp;
  g.lane = lane;
  g.lxi = g.lane & 15;
  g.lx = (float)g.lxi;
  g.px = g.tx * kTile + g.lxi;
  g.x0 = (float)(g.tx * kTile);
  g.y0 = (float)(g.ty * kTile);
#pragma unroll
  for (int s = 0; s < kSlots; ++s) {
    const int lyi = 8 * g.warp + 2 * s + (g.lane >> 4);
    g.ly[s] = (float)lyi;
    g.py[s] = g.ty * kTile + lyi;
    g.inside[s] = g.px < cam.width && g.py[s] < cam.height;
  }
  return g;
}

// Can any point of the rectangle [0,15]^2 - (mx,my) satisfy u^2 + v^2 <= tau, with u = L11 dx + L21 dy, v = L22 dy?
// The minimum of the (convex) form over the rectangle is 0 if it contains the centre, else it lies on one of
// the two edges facing the centre.  `slack` keeps the test conservative against fp32 rounding of either side.
__device__ __forceinline__ bool tile_may_pass(float mx, float my, float L11, float L21, float L22, float qmin) {
  const float tau = -qmin;
  if (!(tau >= 0.f)) return false;  // o G < 1/255 everywhere (also NaN-safe)
  const float xlo = -mx, xhi = 15.0f - mx, ylo = -my, yhi = 15.0f - my;
  const float xn = fminf(fmaxf(0.f, xlo), xhi), yn = fminf(fmaxf(0.f, ylo), yhi);
  const float A = L11 * L11, B = L11 * L21, C = L21 * L21 + L22 * L22;
  // edge dx = xn: dy* = clamp(-B xn / C);  edge dy = yn: dx* = clamp(-B yn / A)
  const float dy1 = fminf(fmaxf(__fdividef(-B * xn, C), ylo), yhi);
  const float dx2 = fminf(fmaxf(__fdividef(-B * yn, A), xlo), xhi);
  // evaluated in the (u,v) form the pixels use, so both sides see the same rounding
  const float u1 = L11 * xn + L21 * dy1, v1 = L22 * dy1;
  const float u2 = L11 * dx2 + L21 * yn, v2 = L22 * yn;
  const float qm = fminf(u1 * u1 + v1 * v1, u2 * u2 + v2 * v2);
  return !(qm > tau * 1.001f + 1e-5f);
}

// Stage up to kBatch list entries.  Candidate c (0 <= c < m) is list position first + c (REVERSE: first - c),
// positions 0-based.  Returns the number of survivors, written in candidate order to s_rec.
// Must be called by all threads of the CTA; ends with a __syncthreads().
// `colour` (may be null): per-primitive (opacity, c0, c1, c2) that replaces float4 #2 of the packed record (the
// auxiliary renders blend other per-primitive quantities through the same kernel).
template <int K, bool REVERSE>
__device__ __forceinline__ int stage_batch(const TileGeom& g, const uint32_t* __restrict__ ids, const float4* __restrict__ packed,
                                           const float4* __restrict__ colour, uint32_t list_begin, int first, int m,
                                           float4* __restrict__ s_rec, uint32_t* __restrict__ s_cnt) {
  constexpr int R4 = packed_floats(K) / 4;
  constexpr int kPer = kBatch / kBlendThreads;
  const int tid = threadIdx.x;
  float4 h0[kPer], h1[kPer];
  uint32_t id[kPer], pos1[kPer], bal[kPer];
  bool keep[kPer];
#pragma unroll
  for (int r = 0; r < kPer; ++r) {
    const int c = r * kBlendThreads + tid;
    keep[r] = false;
    id[r] = 0; pos1[r] = 0;
    if (c < m) {
      const int p = REVERSE ? first - c : first + c;
      pos1[r] = (uint32_t)p + 1u;
      id[r] = __ldg(ids + list_begin + (uint32_t)p);
    }
  }
#pragma unroll
  for (int r = 0; r < kPer; ++r) {
    const int c = r * kBlendThreads + tid;
    if (c < m) {
      const float4 a = __ldg(packed + (size_t)id[r] * R4);
      const float4 l = __ldg(packed + (size_t)id[r] * R4 + 1);
      // mean relative to the tile origin: (hi - origin) + lo
      const float mx = __fadd_rn(__fsub_rn(a.x, g.x0), a.z);
      const float my = __fadd_rn(__fsub_rn(a.y, g.y0), a.w);
      h0[r] = make_float4(mx, my, l.x, l.y);
      h1[r] = make_float4(l.z, l.w, __uint_as_float(pos1[r]), __uint_as_float(id[r]));
      keep[r] = tile_may_pass(mx, my, l.x, l.y, l.z, l.w);
    }
    bal[r] = __ballot_sync(kFull, keep[r]);
    if (g.lane == 0) s_cnt[r * (kBlendThreads / 32) + g.warp] = __popc(bal[r]);
  }
  __syncthreads();
  constexpr int kGroups = kPer * (kBlendThreads / 32);
  uint32_t total = 0;
  uint32_t base[kPer];
#pragma unroll
  for (int r = 0; r < kPer; ++r) base[r] = 0;
#pragma unroll
  for (int q = 0; q < kGroups; ++q) {
#pragma unroll
    for (int r = 0; r < kPer; ++r)
      if (q == r * (kBlendThreads / 32) + g.warp) base[r] = total;
    total += s_cnt[q];
  }
  const uint32_t lt = (1u << g.lane) - 1u;
#pragma unroll
  for (int r = 0; r < kPer; ++r) {
    if (keep[r]) {
      const uint32_t slot = base[r] + __popc(bal[r] & lt);
      s_rec[slot * R4] = h0[r];
      s_rec[slot * R4 + 1] = h1[r];
    }
  }
  __syncthreads();
  // tails of the survivors (colour, frequencies, weights)
  constexpr int T4 = R4 - 2;
  for (int c = tid; c < (int)total * T4; c += kBlendThreads) {
    const int rec = c / T4, ch = 2 + (c - rec * T4);
    const uint32_t pid = __float_as_uint(s_rec[rec * R4 + 1].w);
    s_rec[rec * R4 + ch] = (ch == 2 && colour) ? __ldg(colour + pid) : __ldg(packed + (size_t)pid * R4 + ch);
  }
  __syncthreads();
  return (int)total;
}

// ---- one primitive at one pixel ---------------------------------------------------------------------

// Quadratic form of the envelope from the packed Cholesky factor, in base 2: G = 2^q, q = -(u^2 + v^2) <= 0  (Eq.3 :101);
// ux = L11 * dx is shared by the 4 slots of a thread.
__device__ __forceinline__ float envelope_q(float ux, float L21, float L22, float dy, float& u, float& v) {
  u = __fmaf_rn(L21, dy, ux);
  v = __fmul_rn(L22, dy);
  return -__fmaf_rn(u, u, __fmul_rn(v, v));
}

// G = 2^q for the base-2 exponent of the packed record (q in [-8, 0]: never denormal)
__device__ __forceinline__ float envelope_exp2(float q) {
  float g;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(g) : "f"(q));
  return g;
}

template <int K>
struct Modulation {
  float M;
  float cs[K > 0 ? K : 1], sn[K > 0 ? K : 1];
};

// Per-entry part of the modulation, shared by the 4 pixels of a thread (same column): base = 1 - sum w, and the
// x part of every phase.
template <int K>
struct ModulationEntry {
  float base;
  float phx[K > 0 ? K : 1];
};
template <int K>
__device__ __forceinline__ void modulation_entry(const float* __restrict__ tail, float dx, ModulationEntry<K>& m) {
  float b = 1.0f;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    b = __fsub_rn(b, tail[2 * K + k]);
    m.phx[k] = __fmul_rn(tail[2 * k], dx);
  }
  m.base = b;
}

// M = (1 - sum w) + sum w cos(2 pi f2D . d)   (Eq.12 bracket).  tail = staged (2 pi f2D, omega); the phase is in
// radians and goes to the MUFU unit directly (its own range reduction works in turns: measured error
// 1.2e-7 |phase|).
template <int K, bool WANT_SIN>
__device__ __forceinline__ void modulation(const float* __restrict__ tail, const ModulationEntry<K>& m, float dy, Modulation<K>& e) {
  float M = m.base;
#pragma unroll
  for (int k = 0; k < K; ++k) {
    const float ph = __fmaf_rn(tail[2 * k + 1], dy, m.phx[k]);
    e.cs[k] = __cosf(ph);
    if (WANT_SIN) e.sn[k] = __sinf(ph);
    M = __fmaf_rn(tail[2 * K + k], e.cs[k], M);
  }
  e.M = M;
}

// copy the staged tail (3K floats, padded to float4) into registers
template <int K>
__device__ __forceinline__ void load_tail(const float4* __restrict__ rec, float (&tail)[K > 0 ? 4 * ((3 * K + 3) / 4) : 1]) {
  constexpr int T4 = (3 * K + 3) / 4;
#pragma unroll
  for (int i = 0; i < T4; ++i) {
    const float4 v = rec[3 + i];
    tail[4 * i] = v.x; tail[4 * i + 1] = v.y; tail[4 * i + 2] = v.z; tail[4 * i + 3] = v.w;
  }
}

}  // namespace gabsplat
