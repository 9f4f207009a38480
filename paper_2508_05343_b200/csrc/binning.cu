// S2 / K2-K5: tile binning.  (PAPER.md:103 "sorted by depth", :160 "tile-based rasterizer".)
// The result is the list of (primitive, tile) instances ordered by the 64-bit key (tile << 32) | bits(depth),
// ties by primitive index -- exactly what a stable LSD radix sort of the keys on one-byte digits gives -- plus
// the [start,end) range of every tile.  The depth digits are sorted on the visible primitives, not on the D >> N
// instances; the tile digit then takes one more stable pass:
//   A   (bits(depth), index) of the n_vis visible primitives, compacted in index order, ordered by (depth, index):
//       binned into depth buckets and ranked inside their bucket (3 launches), or -- a bucket too large -- by 4
//       stable one-byte passes -> `order`: visible primitives front to back, ties by index
//   K2  inclusive prefix over that order of the placement cost (B') or of tiles_touched (B) -> offsets (and D for B)
//   B'  images of at most 26000 tiles: ONE stable counting pass on the whole tile id -- per-(tile, chunk) counts,
//       their prefix (tile ranges and D fall out of it), then every instance id written once at its final slot;
//       the 64-bit keys (tile | depth) are written by a coalesced pass if the caller wants them
//   B   larger images: K3 one (tile,id) per (primitive, tile of its rectangle), emitted in depth order, row-major
//       over the rectangle; ceil(tile_bits / 8) stable one-byte passes on the tile id over the D instances, the
//       last one writing the 64-bit key and the id; K5 [start,end) of every tile from the sorted keys
// LSD order is preserved: digits 0-3 (depth) before digits 4.. (tile), every pass stable.  Everything is
// integer work; the result must equal std::stable_sort of the 64-bit keys bit for bit.
// The instance count D lives on the device: every kernel is launched on a grid sized from the caller's
// capacity and returns early past D, so the whole stage runs without a host round trip.
#include <algorithm>

#include "common.cuh"

namespace gabsplat {
namespace {

typedef uint32_t u32;
typedef uint64_t u64;

// ------------------------------------------------------------------------------------------------
// Device-wide prefix sum of u32 (three launches: block sums, scan of the sums, block scans).
// GATHER: element i of the input is in[idx[i]].
// ------------------------------------------------------------------------------------------------
// radix passes: pairs per CTA (declared here: depth_keys_kernel bins its output by sort tile)
constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;  // 4096 pairs per block
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kSmallItems = 16;  // depth passes over the visible primitives (4 was measured slower: more CTAs to sum over)
constexpr int kSmallTile = kSortThreads * kSmallItems;

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;  // 4096 elements per block

__device__ __forceinline__ u32 warp_inclusive_scan(u32 v, int lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const u32 o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}

// Exclusive scan of one value per thread over a block of kScanThreads; returns the exclusive prefix and
// writes the block total to *total.
__device__ __forceinline__ u32 block_exclusive_scan(u32 v, u32* total) {
  __shared__ u32 warp_sums[kScanThreads / 32];
  __shared__ u32 block_total;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const u32 inc = warp_inclusive_scan(v, lane);
  if (lane == 31) warp_sums[w] = inc;
  __syncthreads();
  if (w == 0) {
    const u32 s = lane < kScanThreads / 32 ? warp_sums[lane] : 0;
    const u32 si = warp_inclusive_scan(s, lane);
    if (lane < kScanThreads / 32) warp_sums[lane] = si - s;
    if (lane == kScanThreads / 32 - 1) block_total = si;
  }
  __syncthreads();
  const u32 r = warp_sums[w] + inc - v;
  *total = block_total;
  __syncthreads();
  return r;
}

template <bool GATHER>
__device__ __forceinline__ void scan_load_raw(const u32* __restrict__ in, const u32* __restrict__ idx, u32 base, u32 n,
                                              u32 (&v)[kScanItems]);

// Estimated cost of placing a primitive of t tiles (tile_place_kernel): a fixed part, and per tile ~6x less
// when the primitive is a step of its own (more than `thr` tiles: appended directly) than when it shares a step.
__device__ __forceinline__ u32 place_cost(u32 t, u32 thr) { return 24u + (t > thr ? t / 6u : t); }

// cost_thr != 0: the scanned value is place_cost(in[.], cost_thr) instead of in[.]
template <bool GATHER>
__device__ __forceinline__ void scan_load(const u32* __restrict__ in, const u32* __restrict__ idx, u32 base, u32 n,
                                          u32 cost_thr, u32 (&v)[kScanItems]) {
  scan_load_raw<GATHER>(in, idx, base, n, v);
  if (cost_thr) {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) v[j] = base + j < n ? place_cost(v[j], cost_thr) : 0u;
  }
}

template <bool GATHER>
__device__ __forceinline__ void scan_load_raw(const u32* __restrict__ in, const u32* __restrict__ idx, u32 base, u32 n,
                                              u32 (&v)[kScanItems]) {
  if (base + kScanItems <= n) {
    const uint4* p = reinterpret_cast<const uint4*>((GATHER ? idx : in) + base);
#pragma unroll
    for (int j = 0; j < kScanItems / 4; ++j) {
      const uint4 x = p[j];
      v[4 * j] = x.x; v[4 * j + 1] = x.y; v[4 * j + 2] = x.z; v[4 * j + 3] = x.w;
    }
    if (GATHER) {
#pragma unroll
      for (int j = 0; j < kScanItems; ++j) v[j] = __ldg(in + v[j]);
    }
  } else {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) v[j] = base + j < n ? (GATHER ? __ldg(in + idx[base + j]) : in[base + j]) : 0;
  }
}

template <bool GATHER>
__global__ void __launch_bounds__(kScanThreads) scan_block_sums(const u32* __restrict__ in, const u32* __restrict__ idx, u32 n,
                                                                 const u32* __restrict__ n_dev, u32 cost_thr, u32* __restrict__ sums) {
  pdl_wait();
  if (n_dev) n = min(n, *n_dev);  // the element count lives on the device (n is its host-side bound)
  const u32 base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  u32 v[kScanItems];
  scan_load<GATHER>(in, idx, base, n, cost_thr, v);
  u32 s = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) s += v[j];
  u32 total;
  block_exclusive_scan(s, &total);
  if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

// One block: exclusive scan of sums[0..nb) in place; grand total to *total_out (may be null).
__global__ void __launch_bounds__(kScanThreads) scan_of_sums(u32* __restrict__ sums, u32 nb, u32* __restrict__ total_out) {
  u32 carry = 0;
  for (u32 base = 0; base < nb; base += kScanThreads) {
    const u32 i = base + threadIdx.x;
    const u32 v = i < nb ? sums[i] : 0;
    u32 total;
    const u32 ex = block_exclusive_scan(v, &total);
    if (i < nb) sums[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}

// SELFSUM: `sums` holds the raw block sums and every CTA adds up those of the CTAs before it itself (a few hundred
// at most): the scan is two launches; the last CTA writes the grand total.
template <bool INCLUSIVE, bool GATHER, bool SELFSUM>
__global__ void __launch_bounds__(kScanThreads) scan_apply(const u32* __restrict__ in, const u32* __restrict__ idx, u32 n,
                                                            const u32* __restrict__ n_dev, u32 cost_thr,
                                                            const u32* __restrict__ sums, u32* __restrict__ out,
                                                            u32* __restrict__ total_out) {
  pdl_wait();
  if (n_dev) n = min(n, *n_dev);
  u32 before = 0;
  if (SELFSUM) {
    u32 acc = 0;
    for (u32 b = threadIdx.x; b < blockIdx.x; b += kScanThreads) acc += __ldg(sums + b);
    u32 tot;
    block_exclusive_scan(acc, &tot);
    before = tot;
  } else {
    before = sums[blockIdx.x];
  }
  const u32 base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  u32 v[kScanItems];
  scan_load<GATHER>(in, idx, base, n, cost_thr, v);
  u32 s = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) s += v[j];
  u32 total;
  u32 run = block_exclusive_scan(s, &total) + before;
  if (SELFSUM && total_out && blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) *total_out = before + total;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    const u32 e = run;
    run += v[j];
    v[j] = INCLUSIVE ? run : e;
  }
  if (base + kScanItems <= n) {
    uint4* q = reinterpret_cast<uint4*>(out + base);
#pragma unroll
    for (int j = 0; j < kScanItems / 4; ++j) q[j] = make_uint4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) if (base + j < n) out[base + j] = v[j];
  }
}

inline u32 scan_blocks(u32 n) { return (n + kScanTile - 1) / kScanTile; }

// sums must hold scan_blocks(n) u32.  in/out/idx must be 16-byte aligned.  in == out is allowed (not with GATHER).
template <bool INCLUSIVE, bool GATHER>
void device_scan(const u32* in, const u32* idx, u32* out, u32 n, const u32* n_dev, u32 cost_thr, u32* sums, u32* total_out,
                 cudaStream_t st) {
  const u32 nb = scan_blocks(n);
  if (nb == 0) {
    scan_of_sums<<<1, kScanThreads, 0, st>>>(sums, 0, total_out);
    launched();
    return;
  }
  launch_pdl(scan_block_sums<GATHER>, nb, kScanThreads, 0, st, in, idx, n, n_dev, cost_thr, sums);
  if (nb <= 2048) {
    launch_pdl(scan_apply<INCLUSIVE, GATHER, true>, nb, kScanThreads, 0, st, in, idx, n, n_dev, cost_thr, sums, out, total_out);
    launched(2);
    return;
  }
  scan_of_sums<<<1, kScanThreads, 0, st>>>(sums, nb, total_out);
  launch_pdl(scan_apply<INCLUSIVE, GATHER, false>, nb, kScanThreads, 0, st, in, idx, n, n_dev, cost_thr, sums, out, (u32*)nullptr);
  launched(3);
}

// ------------------------------------------------------------------------------------------------
// A: depth keys of the primitives.  Culled primitives (tiles_touched == 0) sort to the end.
// ------------------------------------------------------------------------------------------------
// One CTA per GABSPLAT_CHUNK consecutive primitives (the chunks of the projection kernel, which left the
// number of visible primitives of every chunk in chunk_visible): the visible primitives are compacted in
// index order -- (bits(depth), index) pairs at [sum of the earlier chunks' counts, ...) -- so that the depth
// passes sort n_vis pairs, not N.
// The depth order is found by BUCKETS when the depths spread (they do in any real scene): the visible primitives
// are binned by (bits(depth) - kmin) >> shift into at most kBuckets bins over the range [kmin, kmax] the projection
// recorded per chunk; a bucket's pairs are gathered (in any order), and every pair finds its place inside its bucket
// by counting the bucket's smaller (depth, index) pairs -- the lexicographic order IS the stable order, so no pass has
// to preserve anything.  Three single-wave launches (histogram with the compaction, scatter, rank) replace the
// compaction and four stable one-byte passes.  A bucket of more than kBucketLimit pairs (thousands of primitives at
// one depth), or buckets so uneven that the ranking would cost more than kRankBudget comparisons per pair, would make
// the quadratic ranking slow: sort_flag is then set and the four radix passes, which are always launched and
// otherwise return at once, sort the compacted pairs instead.
constexpr u32 kBuckets = 8192;
constexpr u32 kBucketLimit = 4096;
constexpr u32 kRankBudget = 256;   // comparisons per pair, on average, the quadratic ranking may cost

struct DepthRange { u32 kmin, shift; };
__device__ __forceinline__ u32 bucket_of(u32 key, const DepthRange& r) { return (key - r.kmin) >> r.shift; }

// kmin / shift from the per-chunk ranges the projection left behind chunk_visible's counts (every CTA computes them itself)
__device__ __forceinline__ DepthRange depth_range(const u32* __restrict__ chunk_visible, u32 nchunks) {
  __shared__ u32 s_min[8], s_max[8];
  u32 lo = 0xffffffffu, hi = 0u;
  for (u32 c = threadIdx.x; c < nchunks; c += 256) {
    lo = min(lo, __ldg(chunk_visible + nchunks + c));
    hi = max(hi, __ldg(chunk_visible + 2 * nchunks + c));
  }
  lo = __reduce_min_sync(0xffffffffu, lo);
  hi = __reduce_max_sync(0xffffffffu, hi);
  if ((threadIdx.x & 31) == 0) { s_min[threadIdx.x >> 5] = lo; s_max[threadIdx.x >> 5] = hi; }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < 8; ++j) { lo = min(lo, s_min[j]); hi = max(hi, s_max[j]); }
  __syncthreads();
  DepthRange r;
  r.kmin = lo;
  const u32 span = hi >= lo ? hi - lo : 0u;
  const int bits = 32 - __clz((int)span);           // span < 2^bits
  r.shift = (u32)max(0, bits - 13);                 // (span >> shift) < kBuckets = 2^13
  return r;
}

__global__ void __launch_bounds__(256) depth_keys_kernel(int N, const u32* __restrict__ tiles_touched,
                                                         const float* __restrict__ depth, const u32* __restrict__ chunk_visible,
                                                         u32* __restrict__ keys, u32* __restrict__ vals, u32* __restrict__ n_vis,
                                                         u32* __restrict__ table0, u32* __restrict__ bucket_cnt,
                                                         u32* __restrict__ slots, DepthRange* __restrict__ range_out) {
  pdl_wait();
  __shared__ u32 s_part[8], s_off;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const DepthRange rg = depth_range(chunk_visible, gridDim.x);
  if (blockIdx.x == 0 && threadIdx.x == 0) *range_out = rg;
  u32 acc = 0;
  for (u32 c = threadIdx.x; c < blockIdx.x; c += 256) acc += __ldg(chunk_visible + c);
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
  if (lane == 0) s_part[w] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    u32 t = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) t += s_part[j];
    s_off = t;
  }
  __syncthreads();
  // the chunk's four rounds of 256 primitives at once: one vote and one exchange of the warp counts for all of them,
  // then every load and every atomic of the thread is in flight before the first result is needed
  constexpr int ROUNDS = GABSPLAT_CHUNK / 256;
  __shared__ u32 s_cnt[ROUNDS][8];
  const int base = blockIdx.x * GABSPLAT_CHUNK;
  bool vis[ROUNDS];
  u32 bal[ROUNDS];
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    const int i = base + r * 256 + (int)threadIdx.x;
    vis[r] = i < N && tiles_touched[i] != 0;
  }
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    bal[r] = __ballot_sync(0xffffffffu, vis[r]);
    if (lane == 0) s_cnt[r][w] = (u32)__popc(bal[r]);
  }
  __syncthreads();
  u32 run = s_off, pos[ROUNDS], key[ROUNDS], slot[ROUNDS];
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    u32 before = 0, total = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { const u32 c = s_cnt[r][j]; before += j < w ? c : 0u; total += c; }
    pos[r] = run + before + (u32)__popc(bal[r] & ((1u << lane) - 1u));
    run += total;
  }
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) key[r] = vis[r] ? __float_as_uint(depth[base + r * 256 + (int)threadIdx.x]) : 0u;
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r)
    slot[r] = vis[r] ? atomicAdd(&bucket_cnt[bucket_of(key[r], rg)], 1u) : 0u;  // arrival number = the pair's slot in its bucket
#pragma unroll
  for (int r = 0; r < ROUNDS; ++r) {
    if (vis[r]) {
      keys[pos[r]] = key[r];
      vals[pos[r]] = (u32)(base + r * 256 + (int)threadIdx.x);
      atomicAdd(&table0[(pos[r] / kSmallTile) * 256u + (key[r] & 255u)], 1u);  // histogram of the first radix pass, per sort tile
      slots[pos[r]] = slot[r];
    }
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) *n_vis = run;
}

// Gathers the compacted pairs by bucket (slot inside the bucket = the arrival number depth_keys_kernel's histogram
// atomic returned): a CTA per kScatterTile pairs.  Every CTA scans the bucket counts itself (32
// per thread); CTA 0 leaves the bucket starts and the path decision for the kernels that follow.
constexpr int kScatterItems = 4;
constexpr int kScatterTile = 256 * kScatterItems;
__global__ void __launch_bounds__(256) bucket_scatter_kernel(const u32* __restrict__ kin, const u32* __restrict__ vin,
                                                             u32* __restrict__ kout, u32* __restrict__ vout,
                                                             const u32* __restrict__ n_vis_p, const u32* __restrict__ bucket_cnt,
                                                             const u32* __restrict__ slots, u32* __restrict__ bucket_base,
                                                             u32* __restrict__ sort_flag, const DepthRange* __restrict__ range) {
  pdl_wait();
  // bucket starts, one padding word per 32 (a thread scans a run of 32 consecutive counts: without the padding the 256
  // runs start in the same bank)
  __shared__ u32 s_base[kBuckets + kBuckets / 32];
  __shared__ u32 s_big;
  __shared__ unsigned long long s_sq;
  auto at = [](u32 i) { return i + (i >> 5); };
  const u32 n = *n_vis_p;
  const u32 start = blockIdx.x * kScatterTile;
  if (start >= n && blockIdx.x != 0) return;
  const DepthRange rg = *range;
  if (threadIdx.x == 0) { s_big = 0; s_sq = 0; }
  __syncthreads();
  // this thread's pairs and their buckets first: the loads are in flight while the counts are scanned
  u32 key[kScatterItems], val[kScatterItems], slot[kScatterItems];
#pragma unroll
  for (int i = 0; i < kScatterItems; ++i) {
    const u32 j = start + (u32)i * 256u + threadIdx.x;
    key[i] = j < n ? __ldg(kin + j) : 0u;
    val[i] = j < n ? __ldg(vin + j) : 0u;
    slot[i] = j < n ? __ldg(slots + j) : 0u;
  }
  constexpr int PER = kBuckets / 256;
  u32 c[PER], sum = 0, mx = 0;
  unsigned long long sq = 0;  // the ranking work: sum of the squared bucket sizes
#pragma unroll
  for (int j = 0; j < PER; j += 4) {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(bucket_cnt + threadIdx.x * PER + j));
    c[j] = v.x; c[j + 1] = v.y; c[j + 2] = v.z; c[j + 3] = v.w;
  }
#pragma unroll
  for (int j = 0; j < PER; ++j) { sum += c[j]; mx = max(mx, c[j]); sq += (unsigned long long)c[j] * c[j]; }
  u32 total;
  u32 run = block_exclusive_scan(sum, &total);
#pragma unroll
  for (int j = 0; j < PER; ++j) { s_base[at(threadIdx.x * PER + j)] = run; run += c[j]; }
  // one huge bucket, or many large ones (more than kRankBudget comparisons per pair on average): the radix passes
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, d);
  if ((threadIdx.x & 31) == 0) atomicAdd(&s_sq, sq);
  if (mx > kBucketLimit) atomicOr(&s_big, 1u);
  __syncthreads();
  if (threadIdx.x == 0 && s_sq > (unsigned long long)kRankBudget * n) s_big = 1u;
  __syncthreads();
  if (blockIdx.x == 0) {
#pragma unroll
    for (int j = 0; j < PER; ++j) bucket_base[threadIdx.x * PER + j] = s_base[at(threadIdx.x * PER + j)];
    if (threadIdx.x == 0) *sort_flag = s_big;
  }
  if (s_big) return;  // the radix passes sort the compacted pairs instead
#pragma unroll
  for (int i = 0; i < kScatterItems; ++i) {
    const u32 j = start + (u32)i * 256u + threadIdx.x;
    if (j < n) {
      const u32 pos = s_base[at(bucket_of(key[i], rg))] + slot[i];
      kout[pos] = key[i];
      vout[pos] = val[i];
    }
  }
}

// place of every pair inside its bucket = the number of the bucket's pairs that are smaller by (depth bits, index)
__global__ void __launch_bounds__(256) bucket_rank_kernel(const u32* __restrict__ kin, const u32* __restrict__ vin,
                                                          u32* __restrict__ kout, u32* __restrict__ vout,
                                                          const u32* __restrict__ n_vis_p, const u32* __restrict__ bucket_cnt,
                                                          const u32* __restrict__ bucket_base, const u32* __restrict__ sort_flag,
                                                          const DepthRange* __restrict__ range) {
  pdl_wait();
  if (*sort_flag) return;
  const u32 p = blockIdx.x * 256u + threadIdx.x;
  if (p >= *n_vis_p) return;
  const DepthRange rg = *range;
  const u32 key = kin[p], val = vin[p];
  const u32 b = bucket_of(key, rg);
  const u32 lo = __ldg(bucket_base + b), cnt = __ldg(bucket_cnt + b);
  u32 rank = 0;
#pragma unroll 8
  for (u32 q = lo; q < lo + cnt; ++q) {
    const u32 kq = __ldg(kin + q), vq = __ldg(vin + q);
    rank += (kq < key || (kq == key && vq < val)) ? 1u : 0u;
  }
  kout[lo + rank] = key;
  vout[lo + rank] = val;
}

// ------------------------------------------------------------------------------------------------
// K3: duplicate, balanced by OUTPUT: one block per kDupChunk consecutive instances (in depth order the
// front-most primitives cover thousands of tiles each and sit next to each other, so a block per 256
// primitives would serialise them).  The block finds the first primitive rank of its chunk with a cooperative
// 256-ary search over `offsets`, stages the chunk's slice of `offsets` / `order` in shared memory, and every
// instance locates its primitive by a binary search there.  Emits the tile id (sort key of stage B) and the
// primitive id; instances of a primitive are row-major over its rectangle.
// ------------------------------------------------------------------------------------------------
constexpr int kDupThreads = 256;
constexpr int kDupChunk = 2048;

__global__ void __launch_bounds__(kDupThreads) duplicate_kernel(const u32* __restrict__ n_vis_p, int tiles_x, const u32* __restrict__ order,
                                                               const u32* __restrict__ offsets,
                                                               const int4* __restrict__ rect,
                                                               const u32* __restrict__ num_instances, u64 capacity,
                                                               u32* __restrict__ tiles_out, u32* __restrict__ ids_out) {
  __shared__ u32 s_incl[kDupChunk];
  __shared__ u32 s_id[kDupChunk];
  __shared__ u32 s_lo, s_hi, s_cnt[kDupThreads / 32];
  const u32 D = *num_instances;
  if ((u64)D > capacity) return;
  const int N = (int)*n_vis_p;  // ranks of the depth order (visible primitives only)
  const u32 g0 = blockIdx.x * kDupChunk;
  if (g0 >= D) return;
  const u32 n = min((u32)kDupChunk, D - g0);
  // r_lo = first rank r with offsets[r] > g0 (upper bound).  Invariant lo <= r_lo <= hi; every step probes 256
  // evenly spaced ranks: the predicate offsets[p] <= g0 holds exactly for p < r_lo, so the true probes are a prefix
  if (threadIdx.x == 0) { s_lo = 0; s_hi = (u32)N; }
  __syncthreads();
  while (true) {
    const u32 lo = s_lo, hi = s_hi;
    if (lo >= hi) break;
    const u32 step = (hi - lo + kDupThreads - 1) / kDupThreads;
    const u32 p = lo + threadIdx.x * step;
    const bool le = p < hi && __ldg(offsets + p) <= g0;
    const u32 bal = __ballot_sync(0xffffffffu, le);
    if ((threadIdx.x & 31) == 0) s_cnt[threadIdx.x >> 5] = __popc(bal);
    __syncthreads();
    if (threadIdx.x == 0) {
      u32 c = 0;
#pragma unroll
      for (int w = 0; w < kDupThreads / 32; ++w) c += s_cnt[w];
      if (c == 0) {
        s_hi = lo;  // offsets[lo] > g0
      } else {
        s_lo = lo + (c - 1) * step + 1;   // probe c-1 holds
        s_hi = min(hi, lo + c * step);    // probe c (if any) does not
      }
    }
    __syncthreads();
  }
  const u32 r_lo = s_lo;
  const u32 prev0 = r_lo ? __ldg(offsets + r_lo - 1) : 0u;  // instances before rank r_lo
  // at most n ranks start inside the chunk (every rank after the first that owns an instance here)
  for (u32 j = threadIdx.x; j < n; j += kDupThreads) {
    const u32 r = r_lo + j;
    s_incl[j] = r < (u32)N ? __ldg(offsets + r) : 0xffffffffu;
    s_id[j] = r < (u32)N ? __ldg(order + r) : 0u;
  }
  __syncthreads();
  for (u32 e = threadIdx.x; e < n; e += kDupThreads) {
    const u32 g = g0 + e;
    // first j with s_incl[j] > g
    u32 lo = 0, hi = n - 1;
    while (lo < hi) {
      const u32 mid = (lo + hi) >> 1;
      if (s_incl[mid] > g) hi = mid; else lo = mid + 1;
    }
    const u32 id = s_id[lo];
    const int4 rc = __ldg(rect + id);
    const u32 first = lo ? s_incl[lo - 1] : prev0;
    const u32 local = g - first;
    const u32 w = (u32)(rc.z - rc.x);
    const u32 row = local / w, col = local - row * w;
    tiles_out[g] = (u32)(rc.y + row) * (u32)tiles_x + (u32)rc.x + col;
    ids_out[g] = id;
  }
}

// ------------------------------------------------------------------------------------------------
// One LSD radix pass on the one-byte digit (key >> shift) & 255 of (u32 key, u32 value) pairs: per-block digit
// histogram, scan of the [digit][block] table, stable scatter.  FINAL (last pass of stage B): the output is
// the 64-bit key (key << 32) | gather[value] and the value.
// ------------------------------------------------------------------------------------------------

// BLOCK_MAJOR: table[block][digit] (read back by sort_scatter<., true>); else table[digit][block] (scanned in place)
template <bool BLOCK_MAJOR>
__global__ void __launch_bounds__(kSortThreads) sort_histogram(const u32* __restrict__ keys, const u32* __restrict__ count,
                                                              u32* __restrict__ table, u32 nblocks, int shift) {
  __shared__ u32 hist[kSortWarps][256];
#pragma unroll
  for (int j = 0; j < kSortWarps; ++j) hist[j][threadIdx.x] = 0;
  __syncthreads();
  const u32 D = *count;
  const u32 start = blockIdx.x * kSortTile;
  const int w = threadIdx.x >> 5;
  if (start < D) {
    const u32 n = min((u32)kSortTile, D - start);
    if (n == kSortTile) {
      const uint4* p = reinterpret_cast<const uint4*>(keys + start);
#pragma unroll
      for (int j = 0; j < kSortItems / 4; ++j) {
        const uint4 k = p[j * kSortThreads + threadIdx.x];
        atomicAdd(&hist[w][(k.x >> shift) & 255u], 1u);
        atomicAdd(&hist[w][(k.y >> shift) & 255u], 1u);
        atomicAdd(&hist[w][(k.z >> shift) & 255u], 1u);
        atomicAdd(&hist[w][(k.w >> shift) & 255u], 1u);
      }
    } else {
      for (u32 j = threadIdx.x; j < n; j += kSortThreads) atomicAdd(&hist[w][(keys[start + j] >> shift) & 255u], 1u);
    }
  }
  __syncthreads();
  u32 tot = 0;
#pragma unroll
  for (int j = 0; j < kSortWarps; ++j) tot += hist[j][threadIdx.x];
  if (BLOCK_MAJOR) table[blockIdx.x * 256u + threadIdx.x] = tot;
  else table[threadIdx.x * nblocks + blockIdx.x] = tot;
}

// SELF: the table holds raw per-block counts, block-major; every CTA sums the columns of the blocks before it
// and the digit totals itself (a few dozen blocks when the pairs are the visible primitives): two launches per
// pass instead of five.  Otherwise the table holds the exclusive scan of the digit-major counts.
// ITEMS pairs per thread: 16 on the instance-sized lists; 4 on the visible primitives, where a pass is a single
// wave of CTAs and its time is one CTA's latency (4 ranking rounds instead of 16)
template <bool FINAL, bool SELF, int ITEMS = kSortItems>
__global__ void __launch_bounds__(kSortThreads) sort_scatter(const u32* __restrict__ kin, const u32* __restrict__ vin,
                                                            u32* __restrict__ kout, u32* __restrict__ vout,
                                                            u64* __restrict__ kout64, const u32* __restrict__ gather,
                                                            const u32* __restrict__ count, const u32* __restrict__ table,
                                                            u32 nblocks, int shift, u32* __restrict__ table_next,
                                                            const u32* __restrict__ run_flag) {
  pdl_wait();
  if (run_flag && *run_flag == 0) return;  // the bucketed depth sort has done the work (see depth_keys_kernel)
  __shared__ u32 warp_hist[kSortWarps][256];
  __shared__ u32 local_base[256];
  __shared__ u32 global_base[256];
  constexpr int TILE = kSortThreads * ITEMS;
  __shared__ u32 skeys[TILE];
  __shared__ u32 svals[TILE];
  const u32 D = *count;
  const u32 start = blockIdx.x * TILE;
  if (start >= D) return;
  const u32 n = min((u32)TILE, D - start);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < kSortWarps; ++j) warp_hist[j][threadIdx.x] = 0;
  __syncthreads();

  // warp w owns the contiguous run [w * 32 * ITEMS, (w+1) * 32 * ITEMS) of the block's tile, visited
  // 32 consecutive pairs at a time: rank order = input order (stability)
  u32 k[ITEMS], v[ITEMS], rank[ITEMS];
  const u32 lt_mask = (1u << lane) - 1u;
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const u32 idx = (u32)w * 32u * ITEMS + (u32)r * 32u + (u32)lane;
    const bool valid = idx < n;
    k[r] = valid ? kin[start + idx] : 0xffffffffu;
    v[r] = valid ? vin[start + idx] : 0;
  }
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const u32 idx = (u32)w * 32u * ITEMS + (u32)r * 32u + (u32)lane;
    const bool valid = idx < n;
    const u32 d = (k[r] >> shift) & 255u;
    // lanes holding the same digit; invalid lanes get a digit value no valid lane can have
#ifdef GS_SORT_MATCH_ANY
    const u32 peers = __match_any_sync(0xffffffffu, valid ? d : 256u);
#else
    // lanes holding the same digit: one vote per digit bit (MATCH.ANY is far slower than 8 VOTEs on sm_100a:
    // ncu showed 60 % of the kernel's stalls waiting on it)
    u32 peers = __ballot_sync(0xffffffffu, valid);
    if (!valid) peers = ~peers;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      const bool bit = (d >> b) & 1u;
      const u32 bal = __ballot_sync(0xffffffffu, bit);
      peers &= bit ? bal : ~bal;
    }
#endif
    u32 prev = 0;
    const int leader = __ffs(peers) - 1;
    if (valid && lane == leader) {
      prev = warp_hist[w][d];
      warp_hist[w][d] = prev + __popc(peers);
    }
    prev = __shfl_sync(0xffffffffu, prev, leader);
    rank[r] = prev + __popc(peers & lt_mask);
    __syncwarp();
  }
  __syncthreads();
  // per digit (one thread each): exclusive prefix over the warps, then over the digits
  {
    const int d = threadIdx.x;
    u32 tot = 0;
#pragma unroll
    for (int j = 0; j < kSortWarps; ++j) {
      const u32 c = warp_hist[j][d];
      warp_hist[j][d] = tot;
      tot += c;
    }
    u32 total;
    const u32 ex = block_exclusive_scan(tot, &total);
    local_base[d] = ex;
    if (SELF) {
      const u32 nact = (D + TILE - 1) / TILE;
      u32 below = 0, all = 0;
#pragma unroll 8
      for (u32 bb = 0; bb < nact; ++bb) {  // independent loads: keep 8 in flight
        const u32 c = __ldg(table + bb * 256u + (u32)d);
        all += c;
        below += bb < blockIdx.x ? c : 0u;
      }
      u32 gtotal;
      global_base[d] = block_exclusive_scan(all, &gtotal) + below;
    } else {
      global_base[d] = table[(u32)d * nblocks + blockIdx.x];
    }
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < ITEMS; ++r) {
    const u32 idx = (u32)w * 32u * ITEMS + (u32)r * 32u + (u32)lane;
    if (idx < n) {
      const u32 d = (k[r] >> shift) & 255u;
      const u32 pos = local_base[d] + warp_hist[w][d] + rank[r];
      skeys[pos] = k[r];
      svals[pos] = v[r];
    }
  }
  __syncthreads();
  for (u32 j = threadIdx.x; j < n; j += kSortThreads) {
    const u32 key = skeys[j];
    const u32 val = svals[j];
    const u32 d = (key >> shift) & 255u;
    const u32 dst = global_base[d] + (j - local_base[d]);
    if (FINAL) kout64[dst] = ((u64)key << 32) | (u64)__ldg(gather + val);
    else kout[dst] = key;
    vout[dst] = val;
    // SELF: the next pass's per-tile histogram (of this pass's output arrangement), so that a pass is one launch
    if (SELF && table_next) atomicAdd(&table_next[(dst / TILE) * 256u + ((key >> (shift + 8)) & 255u)], 1u);
  }
}

// ------------------------------------------------------------------------------------------------
// K5: tile ranges from the sorted keys.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) tile_ranges_kernel(const u64* __restrict__ keys, const u32* __restrict__ num_instances,
                                                          u64 capacity, uint2* __restrict__ ranges) {
  const u32 D = *num_instances;
  if ((u64)D > capacity) return;
  for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < D; i += gridDim.x * blockDim.x) {
    const u32 tile = (u32)(keys[i] >> 32);
    if (i == 0 || (u32)(keys[i - 1] >> 32) != tile) ranges[tile].x = i;
    if (i + 1 == D || (u32)(keys[i + 1] >> 32) != tile) ranges[tile].y = i + 1;
  }
}

// ------------------------------------------------------------------------------------------------
// Launch order of the blend CTAs: the tiles by descending work (longest processing time first), so that the
// last wave of CTAs is made of the shortest lists (ncu: 9-12 % of the SM cycles of both blend kernels were
// idle in the tail with tiles launched in raster order).  One CTA: max, 256-bucket counting sort by
// work / max; the order inside a bucket is immaterial.
// ------------------------------------------------------------------------------------------------
// MODE 0: work(t) = pairs[t].y - pairs[t].x;  1: pairs[t].x + pairs[t].y;  2: ((const u32*)pairs)[t]
// order[] = the items 0..n-1 by descending work(item): one CTA, max, 256-bucket counting sort by work / max
template <typename Work>
__device__ __forceinline__ void block_order_descending(Work work, u32 n, u32* __restrict__ order) {
  __shared__ u32 s_max, s_hist[256], s_base[256];
  if (threadIdx.x == 0) s_max = 0;
  if (threadIdx.x < 256) s_hist[threadIdx.x] = 0;
  __syncthreads();
  u32 mx = 0;
  for (u32 t = threadIdx.x; t < n; t += blockDim.x) mx = max(mx, work(t));
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
  if ((threadIdx.x & 31) == 0) atomicMax(&s_max, mx);
  __syncthreads();
  const float scale = 255.0f / (float)max(s_max, 1u);
  auto bucket = [&](u32 t) { return 255u - min(255u, (u32)((float)work(t) * scale)); };
  for (u32 t = threadIdx.x; t < n; t += blockDim.x) atomicAdd(&s_hist[bucket(t)], 1u);
  __syncthreads();
  if (threadIdx.x < 32) {  // exclusive scan of 256 counts by one warp, 8 per lane
    u32 c[8], tot = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { c[j] = s_hist[threadIdx.x * 8 + j]; tot += c[j]; }
    u32 run = warp_inclusive_scan(tot, threadIdx.x) - tot;
#pragma unroll
    for (int j = 0; j < 8; ++j) { s_base[threadIdx.x * 8 + j] = run; run += c[j]; }
  }
  __syncthreads();
  for (u32 t = threadIdx.x; t < n; t += blockDim.x) order[atomicAdd(&s_base[bucket(t)], 1u)] = t;
}

template <int MODE>
__global__ void __launch_bounds__(1024) tile_order_kernel(const uint2* __restrict__ pairs, u32 ntiles, u32* __restrict__ order) {
  pdl_wait();
  block_order_descending([&](u32 t) -> u32 {
    if (MODE == 2) return reinterpret_cast<const u32*>(pairs)[t];
    const uint2 p = pairs[t];
    return MODE == 1 ? p.x + p.y : p.y - p.x;
  }, ntiles, order);
}

// D in 64 bits on the radix path: the 32-bit prefix sum of tiles_touched wraps at 2^32 instances, and a wrapped
// count could pass every `D > capacity` guard.  total64 (zeroed before) accumulates the tile counts of the visible
// primitives; clamp_count_kernel then overwrites *num_instances with the saturated value.
__global__ void __launch_bounds__(256) instance_total_kernel(int N, const u32* __restrict__ tiles_touched,
                                                              unsigned long long* __restrict__ total64) {
  unsigned long long acc = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) acc += tiles_touched[i];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
  if ((threadIdx.x & 31) == 0 && acc) atomicAdd(total64, acc);
}

__global__ void clamp_count_kernel(u32* sort_count, u32* num_instances, const unsigned long long* total64, u64 capacity) {
  // the sort kernels see 0 instances when the caller's buffers are too small; a count beyond 32 bits saturates
  const unsigned long long D = *total64;
  *num_instances = (u32)min(D, 0xffffffffull);
  *sort_count = (D > capacity || D > 0xffffffffull) ? 0u : (u32)D;
}

// ------------------------------------------------------------------------------------------------
// B': the tile digit in ONE stable counting-sort pass.  The depth-ordered primitive sequence is cut into
// kChunks chunks of equal estimated cost; because a primitive covers a tile at most once, the per-(chunk, tile)
// histogram is simply the number of the chunk's primitives whose rectangle contains the tile:
//   tile_count_kernel   table[chunk][tile] = that number                       (shared-memory histogram per CTA)
//   tile_scan_kernel    table[.][tile] -> exclusive prefix over the chunks; totals[tile]
//   tile_ranges_scan    exclusive prefix of the totals over the tiles -> tile_ranges (+ launch order of the blend)
//   tile_place_kernel   every CTA re-walks its chunk in depth order, kStep primitives at a time, and writes
//                       (tile | depth, id) at  ranges[tile].x + table[chunk][tile] + (rank inside the chunk)
// The rank inside a step is the number of lower-ranked primitives of the step that cover the same tile: the
// step's primitives OR their bit into mask[tile] (shared memory), then every instance counts the bits below
// its own.  Result: exactly the order of a stable sort by tile of the depth-ordered instance sequence, i.e.
// what the one-byte LSD passes on the tile digits produce (kept below as the path for images with more tiles
// than fit in shared memory), at a fraction of the traffic: the instances are written once and never read.
// ------------------------------------------------------------------------------------------------
constexpr int kChunks = 592;       // 4 per SM
constexpr int kPlaceThreads = 256;
constexpr int kStep = 32;          // primitives per step (one mask bit each)
constexpr int kMaxTilesCounting = 26000;  // 2 * 4 B * tiles (and 4 B * (tiles_x+1)(tiles_y+1)) of shared memory must fit in 227 KB

// boundary c of the chunking: the number of ranks r < n_vis whose inclusive cost prefix is <= c * total / kChunks
__device__ __forceinline__ void chunk_bound(const u32* __restrict__ offsets, const u32* __restrict__ n_vis_p,
                                            u32* __restrict__ bounds, u32 c) {
  __shared__ u32 s_lo, s_hi, s_cnt[8];
  const u32 n_vis = *n_vis_p;
  if (n_vis == 0) { if (threadIdx.x == 0) bounds[c] = 0; return; }
  const u64 total = (u64)__ldg(offsets + n_vis - 1);  // offsets = inclusive prefix of place_cost in depth order
  const u64 target = total * c / kChunks;
  if (threadIdx.x == 0) { s_lo = 0; s_hi = n_vis; }
  __syncthreads();
  while (true) {
    const u32 lo = s_lo, hi = s_hi;
    if (lo >= hi) break;
    const u32 step = (hi - lo + 255) / 256;
    const u32 p = lo + threadIdx.x * step;
    const bool le = p < hi && (u64)__ldg(offsets + p) <= target;
    const u32 bal = __ballot_sync(0xffffffffu, le);
    if ((threadIdx.x & 31) == 0) s_cnt[threadIdx.x >> 5] = __popc(bal);
    __syncthreads();
    if (threadIdx.x == 0) {
      u32 k = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) k += s_cnt[w];
      if (k == 0) s_hi = lo;
      else { s_lo = lo + (k - 1) * step + 1; s_hi = min(hi, lo + k * step); }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) bounds[c] = s_lo;
}

// record r of the depth-ordered visible primitives: (id, bits(depth), x0 | y0 << 16, x1 | y1 << 16): what the two
// walks below read, coalesced, instead of chasing order -> rect / depth per primitive
// One launch for two independent jobs: CTAs 0..kChunks compute the chunk boundaries, the others write the records.
inline int record_ctas() { return sm_count() * 4; }
__global__ void __launch_bounds__(256) bounds_records_kernel(const u32* __restrict__ offsets, const u32* __restrict__ order,
                                                             const int4* __restrict__ rect, const float* __restrict__ depth,
                                                             const u32* __restrict__ n_vis_p, u32* __restrict__ bounds,
                                                             uint4* __restrict__ recs) {
  pdl_wait();
  if (blockIdx.x <= kChunks) { chunk_bound(offsets, n_vis_p, bounds, blockIdx.x); return; }
  const u32 n_vis = *n_vis_p;
  for (u32 r = (blockIdx.x - kChunks - 1) * blockDim.x + threadIdx.x; r < n_vis; r += (gridDim.x - kChunks - 1) * blockDim.x) {
    const u32 id = __ldg(order + r);
    const int4 rc = __ldg(rect + id);
    recs[r] = make_uint4(id, __float_as_uint(__ldg(depth + id)), (u32)rc.x | ((u32)rc.y << 16), (u32)rc.z | ((u32)rc.w << 16));
  }
}

// walks the tiles of one rectangle: f(tile) for tile number start, start + stride, ... (row-major in the rectangle);
// tile ids are relative to tile row `ysub`
template <typename F>
__device__ __forceinline__ void for_rect_tiles(u32 xy0, u32 xy1, int tiles_x, int ysub, int start, int stride, F f) {
  const int x0 = (int)(xy0 & 0xffffu), y0 = (int)(xy0 >> 16);
  const int w = (int)(xy1 & 0xffffu) - x0, n = w * ((int)(xy1 >> 16) - y0);
  // floor(a / w) for 0 <= a <= 256 without an integer division: (a + 0.5) / w is at least 0.5 / w away from
  // every integer, far more than the error of the approximate quotient
  const float fw = (float)w;
  int row = __float2int_rz(__fdividef((float)start + 0.5f, fw)), col = start - row * w;
  const int drow = __float2int_rz(__fdividef((float)stride + 0.5f, fw)), dcol = stride - drow * w;
  for (int e = start; e < n; e += stride) {
    f((u32)((y0 - ysub + row) * tiles_x + x0 + col));
    row += drow; col += dcol;
    if (col >= w) { col -= w; ++row; }
  }
}

// table[chunk][tile] = number of the chunk's primitives whose rectangle contains the tile, by a 2D difference
// array in shared memory: four corner updates per primitive, then prefix sums along x and along y.
__global__ void __launch_bounds__(kPlaceThreads) tile_count_kernel(int tiles_x, int tiles_y, const uint4* __restrict__ recs,
                                                                   const u32* __restrict__ bounds, u32* __restrict__ table) {
  pdl_wait();
  extern __shared__ int s_d[];  // [(tiles_y + 1)][(tiles_x + 1)]
  const int sx = tiles_x + 1, sy = tiles_y + 1;
  for (int t = threadIdx.x; t < sx * sy; t += kPlaceThreads) s_d[t] = 0;
  __syncthreads();
  const u32 b0 = bounds[blockIdx.x], b1 = bounds[blockIdx.x + 1];
  for (u32 r = b0 + threadIdx.x; r < b1; r += kPlaceThreads) {
    const uint4 rc = __ldg(recs + r);
    const int x0 = (int)(rc.z & 0xffffu), y0 = (int)(rc.z >> 16), x1 = (int)(rc.w & 0xffffu), y1 = (int)(rc.w >> 16);
    atomicAdd(&s_d[y0 * sx + x0], 1);
    atomicAdd(&s_d[y0 * sx + x1], -1);
    atomicAdd(&s_d[y1 * sx + x0], -1);
    atomicAdd(&s_d[y1 * sx + x1], 1);
  }
  __syncthreads();
  for (int y = threadIdx.x; y < sy; y += kPlaceThreads) {
    int run = 0;
    for (int x = 0; x < sx; ++x) { run += s_d[y * sx + x]; s_d[y * sx + x] = run; }
  }
  __syncthreads();
  for (int x = threadIdx.x; x < sx; x += kPlaceThreads) {
    int run = 0;
    for (int y = 0; y < sy; ++y) { run += s_d[y * sx + x]; s_d[y * sx + x] = run; }
  }
  __syncthreads();
  const int ntiles = tiles_x * tiles_y;
  for (int t = threadIdx.x; t < ntiles; t += kPlaceThreads) {
    const int y = t / tiles_x, x = t - y * tiles_x;
    table[(size_t)blockIdx.x * ntiles + t] = (u32)s_d[y * sx + x];   // chunk-major: a coalesced row per CTA
  }
}

// Exclusive prefix over the chunks of table[chunk][tile], in place, and the total of every tile.  A CTA takes 32
// consecutive tiles (one coalesced 128-byte row segment per chunk) and cuts the chunks into kScanSegs segments, a warp
// each: segment sums first, then the prefixes with the earlier segments' sums added.
constexpr int kScanSegs = 16;
static_assert(kChunks % kScanSegs == 0, "the chunk count must split evenly into scan segments");
__global__ void __launch_bounds__(32 * kScanSegs) tile_scan_kernel(int ntiles, u32* __restrict__ table, u32* __restrict__ totals) {
  pdl_wait();
  constexpr int PER = kChunks / kScanSegs;
  __shared__ u32 s_sum[kScanSegs][32];
  const int lane = threadIdx.x & 31, seg = threadIdx.x >> 5;
  const int t = blockIdx.x * 32 + lane;
  const bool live = t < ntiles;
  u32* col = table + (size_t)seg * PER * ntiles + t;
  u32 v[PER], sum = 0;
#pragma unroll
  for (int i = 0; i < PER; ++i) { v[i] = live ? col[(size_t)i * ntiles] : 0u; sum += v[i]; }
  s_sum[seg][lane] = sum;
  __syncthreads();
  u32 run = 0, all = 0;
#pragma unroll
  for (int j = 0; j < kScanSegs; ++j) { const u32 x = s_sum[j][lane]; run += j < seg ? x : 0u; all += x; }
  if (live) {
#pragma unroll
    for (int i = 0; i < PER; ++i) { col[(size_t)i * ntiles] = run; run += v[i]; }
    if (seg == 0) totals[t] = all;
  }
}

// one CTA: tile_ranges[t] = [start, start + totals[t]) by an exclusive prefix over the tiles ((0,0) for an empty
// tile and for every tile when the instances do not fit the caller's buffers)
__global__ void __launch_bounds__(1024) tile_ranges_scan_kernel(int ntiles, const u32* __restrict__ totals,
                                                               u32* __restrict__ num_instances, u64 capacity,
                                                               uint2* __restrict__ ranges, u32* __restrict__ order,
                                                               const u32* __restrict__ work_hint) {
  pdl_wait();
  // every thread owns a run of consecutive tiles: one block-wide scan of the run sums (64-bit: D may exceed what the
  // 32-bit positions can address), then the starts inside the run
  __shared__ unsigned long long s_warp[32];
  __shared__ unsigned long long s_total;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int per = (ntiles + 1023) / 1024;
  const int t0 = min(ntiles, (int)threadIdx.x * per), t1 = min(ntiles, t0 + per);
  unsigned long long sum = 0;
  for (int t = t0; t < t1; ++t) sum += totals[t];
  unsigned long long inc = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const unsigned long long o = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += o;
  }
  if (lane == 31) s_warp[w] = inc;
  __syncthreads();
  if (w == 0) {
    const unsigned long long x = s_warp[lane];
    unsigned long long xi = x;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const unsigned long long o = __shfl_up_sync(0xffffffffu, xi, d);
      if (lane >= d) xi += o;
    }
    s_warp[lane] = xi - x;
    if (lane == 31) s_total = xi;
  }
  __syncthreads();
  const unsigned long long D = s_total;
  const bool fits = D <= capacity && D <= 0xffffffffull;
  if (threadIdx.x == 0) *num_instances = (u32)min(D, 0xffffffffull);
  u32 start = (u32)(s_warp[w] + inc - sum);
  for (int t = t0; t < t1; ++t) {
    const u32 v = totals[t];
    ranges[t] = (fits && v) ? make_uint2(start, start + v) : make_uint2(0u, 0u);
    start += v;
  }
  __syncthreads();
  // launch order of the forward blend: tiles by descending list length
  // ... or, with a hint from an earlier render of the view, by how far every tile walked its list then (a tile stops
  // when its last pixel saturates, typically long before the end of its list: the list length does not predict it)
  block_order_descending([&](u32 t) -> u32 {
    const u32 n = fits ? totals[t] : 0u;
    return work_hint ? min(n, __ldg(work_hint + t)) : n;
  }, (u32)ntiles, order);
}

// Instances a thread keeps in registers during a step.  Measured (config 3 / 4 / 2 placement, ms): 8: 0.101 / 0.487 /
// 0.064; 4: 0.093 / 0.457; 2: 0.089 / 0.444 / 0.051; 1: 0.088 / 0.437 / 0.050 -- a shared step of 32 primitives rarely
// fills more than one instance per thread, and a primitive of more than kFlat * THREADS tiles takes the direct path.
#ifndef GS_FLAT
#define GS_FLAT 1
#endif
constexpr int kFlat = GS_FLAT;

__device__ __forceinline__ u32 rect_tiles(const uint4& rc) {
  return ((rc.w & 0xffffu) - (rc.z & 0xffffu)) * ((rc.w >> 16) - (rc.z >> 16));
}

// A step is the longest run of consecutive primitives (at most kStep) whose rectangles hold at most
// kFlat * THREADS tiles together, and at least one primitive.
//  * one primitive: its tiles are all different, so the whole CTA appends its id to their lists directly;
//  * several: instance e of the step belongs to thread e % THREADS, which locates it once (binary search in the
//    prefix of the tile counts, then row / column inside the rectangle) and keeps (tile | w << 16) in registers
//    through the three phases: mark (OR bit w into mask[tile]), place (cursor + bits below w), close (the
//    highest bit advances the cursor and clears the mask).
// THREADS: 256, or 1024 when the two per-tile arrays leave room for only two CTAs per SM (keeps 64 warps resident)
template <int THREADS>
__global__ void __launch_bounds__(THREADS, THREADS == 1024 ? 2 : 4) tile_place_kernel(int ntiles, int tiles_x, const uint4* __restrict__ recs,
                                                                   const u32* __restrict__ bounds, const u32* __restrict__ table,
                                                                   const uint2* __restrict__ ranges,
                                                                   const u32* __restrict__ num_instances, u64 capacity,
                                                                   int band_rows, u32* __restrict__ ids) {
  pdl_wait();
  constexpr u32 kStepInstances = kFlat * THREADS;
  // CTA (chunk, band): the chunk's primitives clipped to the band's tile rows [ylo, yhi).  Bands keep the two
  // per-tile arrays small (many CTAs per SM for this latency-bound walk) and, because the CTAs of a band are
  // dispatched together, the stores of a wave of CTAs fall into one window of the tile-major output, where the
  // 4-byte stores of neighbouring chunks merge into whole sectors in L2.
  const u32 tiles_y = (u32)(ntiles / tiles_x);
  const u32 ylo = blockIdx.y * (u32)band_rows, yhi = min(tiles_y, ylo + (u32)band_rows);
  const u32 tile0 = ylo * (u32)tiles_x, nband = (yhi - ylo) * (u32)tiles_x;
  extern __shared__ u32 s_mem[];
  u32* s_pos = s_mem;           // [nband] next free slot of the tile for this chunk
  u32* s_mask = s_mem + nband;  // [nband] bit w set: primitive w of the current step covers the tile
  __shared__ uint4 s_rec[2][kStep];
  __shared__ u32 s_pre[2][kStep + 1];  // exclusive prefix of the tile counts of the step's primitives
  __shared__ int s_m[2];               // primitives in the step
  if ((u64)*num_instances > capacity) return;
  for (u32 t = threadIdx.x; t < nband; t += THREADS) {
    s_pos[t] = ranges[tile0 + t].x + table[(size_t)blockIdx.x * ntiles + tile0 + t];
    s_mask[t] = 0;
  }
  const u32 b0 = bounds[blockIdx.x], b1 = bounds[blockIdx.x + 1];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  // warp 0 stages the step that starts at rank r
  auto stage = [&](int buf, u32 r) {
    const bool have = r + lane < b1;
    uint4 rc = have ? __ldg(recs + r + lane) : make_uint4(0u, 0u, 0u, 0u);
    {  // clip the rectangle to the band; an empty intersection becomes a rectangle of zero rows
      const u32 y0 = min(max(rc.z >> 16, ylo), yhi), y1 = min(max(rc.w >> 16, y0), yhi);
      rc.z = (rc.z & 0xffffu) | (y0 << 16);
      rc.w = (rc.w & 0xffffu) | (y1 << 16);
    }
    const u32 n = have ? rect_tiles(rc) : 0u;
    const u32 inc = warp_inclusive_scan(n, lane);
    const int m = max(1, __popc(__ballot_sync(0xffffffffu, have && inc <= kStepInstances)));
    s_rec[buf][lane] = rc;
    s_pre[buf][lane + 1] = lane < m ? inc : 0xffffffffu;  // the binary search never steps past primitive m - 1
    if (lane == 0) { s_pre[buf][0] = 0; s_m[buf] = m; }
  };
  if (warp == 0 && b0 < b1) stage(0, b0);
  int buf = 0;
  u32 r0 = b0;
  while (r0 < b1) {
    __syncthreads();  // stage(buf) visible; first step: s_pos / s_mask initialised; previous step finished
    const int m = s_m[buf];
    const u32 total = s_pre[buf][m];
    if (warp == 0 && r0 + m < b1) stage(buf ^ 1, r0 + m);  // overlaps the global load with this step
    if (m == 1) {
      const uint4 rc = s_rec[buf][0];
      for_rect_tiles(rc.z, rc.w, tiles_x, (int)ylo, (int)threadIdx.x, THREADS, [&](u32 t) { ids[s_pos[t]++] = rc.x; });
    } else {
      u32 tw[kFlat];
#pragma unroll
      for (int i = 0; i < kFlat; ++i) {
        const u32 e = (u32)i * THREADS + threadIdx.x;
        tw[i] = 0xffffffffu;
        if (e < total) {
          u32 w = 0;
#pragma unroll
          for (int b = kStep / 2; b > 0; b >>= 1) if (s_pre[buf][w + b] <= e) w += b;
          const uint4 rc = s_rec[buf][w];
          const u32 x0 = rc.z & 0xffffu, y0 = rc.z >> 16, wd = (rc.w & 0xffffu) - x0;
          const u32 local = e - s_pre[buf][w];
          const u32 row = (u32)__float2int_rz(__fdividef((float)local + 0.5f, (float)wd));  // local < 8192: exact (the quotient error, ~local * 2^-22 / wd, is far below the 0.5 / wd margin)
          const u32 t = (y0 - ylo + row) * (u32)tiles_x + x0 + (local - row * wd);
          tw[i] = t | (w << 16);
          atomicOr(&s_mask[t], 1u << w);
        }
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < kFlat; ++i) {
        if (tw[i] != 0xffffffffu) {
          const u32 t = tw[i] & 0xffffu, w = tw[i] >> 16;
          ids[s_pos[t] + __popc(s_mask[t] & ((1u << w) - 1u))] = s_rec[buf][w].x;
        }
      }
      __syncthreads();
#pragma unroll
      for (int i = 0; i < kFlat; ++i) {
        if (tw[i] != 0xffffffffu) {
          const u32 t = tw[i] & 0xffffu, w = tw[i] >> 16;
          const u32 mk = s_mask[t];
          if ((mk >> w) == 1u) { s_pos[t] += __popc(mk); s_mask[t] = 0; }
        }
      }
    }
    r0 += m;
    buf ^= 1;
  }
}

// keys[i] = (tile << 32) | bits(depth[ids[i]]) for the sorted instances: a warp per tile, coalesced.  (The blend
// kernels never read the keys; they are the inspectable statement of the order.)
__global__ void __launch_bounds__(256) tile_keys_kernel(int ntiles, const uint2* __restrict__ ranges, const u32* __restrict__ ids,
                                                        const float* __restrict__ depth, u64* __restrict__ keys) {
  pdl_wait();
  // half a CTA (128 threads) per tile, two instances per thread and iteration in flight
  const int t = blockIdx.x * 2 + (threadIdx.x >> 7);
  if (t >= ntiles) return;
  const uint2 rg = ranges[t];
  const u64 hi = (u64)(u32)t << 32;
  for (u32 i = rg.x + (threadIdx.x & 127); i < rg.y; i += 256) {
    const u32 j = i + 128;
    const u32 a = ids[i], b = j < rg.y ? ids[j] : 0u;
    const u32 da = __float_as_uint(__ldg(depth + a)), db = __float_as_uint(__ldg(depth + b));
    keys[i] = hi | (u64)da;
    if (j < rg.y) keys[j] = hi | (u64)db;
  }
}

inline u64 align_up(u64 x, u64 a) { return (x + a - 1) / a * a; }
inline u32 sort_blocks(u64 n) { return (u32)((n + kSortTile - 1) / kSortTile); }

struct Workspace {
  u32* scan_sums;   // scan partials (reused by every scan)
  u32* count_a;     // [1] = N
  u32* count_b;     // [1] = D, or 0 when D > capacity
  u32* table;       // [256][nblocks]
  u32* dtable[4];   // per depth pass: [sort_blocks(N)][256] histograms of that pass's input arrangement
  u32* bucket_cnt;  // [kBuckets] pairs per depth bucket          zeroed together with dtable and sort_flag
  u32* slots;       // [N] slot of every compacted pair inside its bucket
  u32* sort_flag;   // [1] 1: a bucket is too large, the radix passes sort instead
  u32* bucket_base; // [kBuckets] first slot of every bucket
  DepthRange* range;  // bucket mapping of this call
  u32* pk[2];       // stage A key ping-pong [N]
  u32* pv[2];       // stage A value ping-pong [N]; pv[0] ends up holding the depth order
  u32* ik;          // stage B (radix path) alternate keys [capacity]
  u32* iv;          // stage B (radix path) alternate values [capacity]
  u32* n_vis;       // [1] number of visible primitives
  u32* bounds;      // [kChunks + 1] chunk boundaries (ranks in depth order)
  u32* totals;      // [ntiles] instances per tile
  uint4* recs;      // [N] records of the visible primitives in depth order
  u32* chunk_table; // [kChunks][ntiles] per-(chunk, tile) counts, then exclusive prefixes over the chunks
  u64 bytes;
};

inline bool counting_path(int ntiles) { return ntiles <= kMaxTilesCounting; }

Workspace carve(void* base, int N, u64 capacity, int ntiles) {
  const u64 nb = (u64)(sort_blocks(capacity) > sort_blocks((u64)N) ? sort_blocks(capacity) : sort_blocks((u64)N));
  const u64 table_n = (u64)256 * (nb ? nb : 1);
  const u64 sums_n = (u64)scan_blocks((u32)(table_n > (u64)N ? table_n : (u64)N)) + 16;
  u64 off = 0;
  Workspace w;
  char* b = (char*)base;
  auto take = [&](u64 bytes) { char* p = b + off; off = align_up(off + bytes, 256); return p; };
  w.scan_sums = (u32*)take(sums_n * 4);
  w.count_a = (u32*)take(16);
  w.count_b = (u32*)take(16);
  w.table = (u32*)take(table_n * 4);
  {  // contiguous, zeroed by one memset per call
    const u64 one = (u64)256 * (((u64)N + kSmallTile - 1) / kSmallTile + 1);
    u32* base4 = (u32*)take((4 * one + kBuckets + 64) * 4);
    for (int i = 0; i < 4; ++i) w.dtable[i] = base4 + i * one;
    w.bucket_cnt = base4 + 4 * one;
    w.sort_flag = w.bucket_cnt + kBuckets;
  }
  w.bucket_base = (u32*)take((u64)kBuckets * 4);
  w.slots = (u32*)take((u64)N * 4);
  w.range = (DepthRange*)take(sizeof(DepthRange));
  for (int i = 0; i < 2; ++i) { w.pk[i] = (u32*)take((u64)N * 4); w.pv[i] = (u32*)take((u64)N * 4); }
  w.n_vis = (u32*)take(16);
  w.bounds = (u32*)take((kChunks + 1) * 4);
  if (counting_path(ntiles)) {
    w.ik = w.iv = nullptr;
    w.totals = (u32*)take((u64)ntiles * 4);
    w.recs = (uint4*)take((u64)N * 16);
    w.chunk_table = (u32*)take((u64)ntiles * kChunks * 4);
  } else {
    w.totals = w.chunk_table = nullptr;
    w.recs = nullptr;
    w.ik = (u32*)take(capacity * 4);
    w.iv = (u32*)take(capacity * 4);
  }
  w.bytes = off;
  return w;
}

void radix_pass(const u32* kin, const u32* vin, u32* kout, u32* vout, u64* kout64, const u32* gather, const u32* count,
                u32 nblocks, int shift, const Workspace& ws, cudaStream_t st) {
  sort_histogram<false><<<nblocks, kSortThreads, 0, st>>>(kin, count, ws.table, nblocks, shift);
  launched();
  device_scan<false, false>(ws.table, nullptr, ws.table, 256u * nblocks, nullptr, 0u, ws.scan_sums, nullptr, st);
  if (kout64)
    launch_pdl(sort_scatter<true, false>, nblocks, kSortThreads, 0, st, kin, vin, kout, vout, kout64, gather, count, ws.table, nblocks, shift, (u32*)nullptr, (const u32*)nullptr);
  else
    launch_pdl(sort_scatter<false, false>, nblocks, kSortThreads, 0, st, kin, vin, kout, vout, kout64, gather, count, ws.table, nblocks, shift, (u32*)nullptr, (const u32*)nullptr);
  launched();
}

// a pass over the visible primitives: ONE launch -- its per-tile histogram was accumulated by the producer of its
// input (depth_keys_kernel for the first pass, the previous pass's scatter for the others)
void radix_pass_small(const u32* kin, const u32* vin, u32* kout, u32* vout, const u32* count, u32 nblocks, int shift,
                      const u32* table, u32* table_next, const u32* run_flag, cudaStream_t st) {
  launch_pdl(sort_scatter<false, true, kSmallItems>, nblocks, kSortThreads, 0, st, kin, vin, kout, vout, (u64*)nullptr,
             (const u32*)nullptr, count, table, nblocks, shift, table_next, run_flag);
  launched();
}

}  // namespace

cudaError_t launch_tile_order(const uint32_t* pairs, bool sum, int ntiles, uint32_t* order, cudaStream_t st) {
  if (ntiles <= 0) return cudaSuccess;
  if (sum) launch_pdl(tile_order_kernel<1>, 1, 1024, 0, st, reinterpret_cast<const uint2*>(pairs), (u32)ntiles, order);
  else launch_pdl(tile_order_kernel<0>, 1, 1024, 0, st, reinterpret_cast<const uint2*>(pairs), (u32)ntiles, order);
  launched();
  return cudaGetLastError();
}

cudaError_t launch_half_tile_order(const uint32_t* work, int n, uint32_t* order, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  launch_pdl(tile_order_kernel<2>, 1, 1024, 0, st, reinterpret_cast<const uint2*>(work), (u32)n, order);
  launched();
  return cudaGetLastError();
}

bool keys_optional(int ntiles) { return counting_path(ntiles); }

void binning_visible_list(const gabsplat_binning& bin, int N, int ntiles, const uint32_t** order, const uint32_t** n_vis) {
  const Workspace ws = carve(bin.workspace, N, bin.capacity, ntiles);
  *order = ws.pv[0];  // four passes: the depth order ends in the buffer it started in
  *n_vis = ws.n_vis;
}

uint64_t sort_workspace_bytes(int N, uint64_t capacity, int ntiles) { return carve(nullptr, N, capacity, ntiles).bytes; }

cudaError_t launch_bin_sort(int N, const gabsplat_projected& proj, const Camera& cam, const gabsplat_binning& bin,
                            StageTimer& tm, int place_bands, cudaStream_t st) {
  const int ntiles = cam.tiles_x * cam.tiles_y;
  const Workspace ws = carve(bin.workspace, N, bin.capacity, ntiles);
  if (N == 0) {
    cudaMemsetAsync(bin.num_instances, 0, sizeof(u32), st);
    cudaMemsetAsync(bin.tile_ranges, 0, (size_t)ntiles * 2 * sizeof(u32), st);
    return launch_tile_order(bin.tile_ranges, false, ntiles, bin.tile_order, st);
  }
  // A: depth order of the primitives (digits 0-3 of the 64-bit key)
  tm.begin(GABSPLAT_STAGE_DEPTH_SORT, st);
  const u32 nba = (u32)(((u64)N + kSmallTile - 1) / kSmallTile);
  cudaMemsetAsync(ws.dtable[0], 0, ((size_t)4 * 256 * (nba + 1) + kBuckets + 64) * sizeof(u32), st);
  const u32 nchunks = (u32)((N + GABSPLAT_CHUNK - 1) / GABSPLAT_CHUNK);
  launch_pdl(depth_keys_kernel, nchunks, 256, 0, st, N, proj.tiles_touched, proj.depth,
             proj.chunk_visible, ws.pk[0], ws.pv[0], ws.n_vis, ws.dtable[0], ws.bucket_cnt, ws.slots, ws.range);
  // bucketed order: pairs gathered by bucket into pk[1] / pv[1], ranked inside their buckets back into pk[0] / pv[0]
  launch_pdl(bucket_scatter_kernel, (u32)((N + kScatterTile - 1) / kScatterTile), 256, 0, st, ws.pk[0], ws.pv[0], ws.pk[1], ws.pv[1],
             ws.n_vis, ws.bucket_cnt, (const u32*)ws.slots, ws.bucket_base, ws.sort_flag, (const DepthRange*)ws.range);
  launch_pdl(bucket_rank_kernel, (u32)((N + 255) / 256), 256, 0, st, ws.pk[1], ws.pv[1], ws.pk[0], ws.pv[0], ws.n_vis,
             ws.bucket_cnt, ws.bucket_base, ws.sort_flag, ws.range);
  launched(3);
  // ... unless a bucket is too large: then these four stable one-byte passes run (otherwise they return at once)
  for (int p = 0; p < 4; ++p)
    radix_pass_small(ws.pk[p & 1], ws.pv[p & 1], ws.pk[(p & 1) ^ 1], ws.pv[(p & 1) ^ 1], ws.n_vis, nba, 8 * p, ws.dtable[p],
                     p < 3 ? ws.dtable[p + 1] : nullptr, ws.sort_flag, st);
  const u32* order = ws.pv[0];
  tm.end(st);
  // K2 (over the n_vis ranks)
  tm.begin(GABSPLAT_STAGE_SCAN, st);
  // counting path: the scanned value is the estimated placement cost of the primitive (chunks of equal cost;
  // the instance count then comes out of the tile totals); otherwise its tile count (offsets, D)
  const bool counting = counting_path(ntiles) && bin.capacity > 0;
  const int place_threads = 256;
  device_scan<true, true>(proj.tiles_touched, order, bin.offsets, (u32)N, ws.n_vis, counting ? (u32)(kFlat * place_threads) : 0u,
                          ws.scan_sums, counting ? ws.count_a : bin.num_instances, st);
  tm.end(st);
  if (bin.capacity == 0) {
    cudaMemsetAsync(bin.tile_ranges, 0, (size_t)ntiles * 2 * sizeof(u32), st);
    return launch_tile_order(bin.tile_ranges, false, ntiles, bin.tile_order, st);
  }
  if (counting) {
    // B': one counting-sort pass on the whole tile id (see the kernels above)
    const size_t smem_count = (size_t)(cam.tiles_x + 1) * (cam.tiles_y + 1) * sizeof(int);
    if (smem_count > 48 * 1024)
      cudaFuncSetAttribute(tile_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_count);
    const int4* rect = reinterpret_cast<const int4*>(proj.rect);
    uint2* ranges = reinterpret_cast<uint2*>(bin.tile_ranges);
    tm.begin(GABSPLAT_STAGE_DUPLICATE, st);
    launch_pdl(bounds_records_kernel, kChunks + 1 + record_ctas(), 256, 0, st, bin.offsets, order, rect, proj.depth, ws.n_vis,
               ws.bounds, ws.recs);
    launch_pdl(tile_count_kernel, kChunks, kPlaceThreads, smem_count, st, cam.tiles_x, cam.tiles_y, ws.recs, ws.bounds, ws.chunk_table);
    launched(2);
    tm.end(st);
    tm.begin(GABSPLAT_STAGE_RANGES, st);
    launch_pdl(tile_scan_kernel, (ntiles + 31) / 32, 32 * kScanSegs, 0, st, ntiles, ws.chunk_table, ws.totals);
    launch_pdl(tile_ranges_scan_kernel, 1, 1024, 0, st, ntiles, ws.totals, bin.num_instances, bin.capacity, ranges, bin.tile_order,
               bin.tile_work_hint);
    launched(2);
    tm.end(st);
    tm.begin(GABSPLAT_STAGE_SORT, st);
    // bands of at most ~1280 tiles: measured best on both the 4346-tile and the 9840-tile configs
    // (gabsplat_set_place_bands overrides the number of bands: instrumentation for the tests)
    u64 nbands = std::max<u64>(1, ((u64)ntiles + 1279) / 1280);
    if (place_bands > 0) nbands = (u64)place_bands;
    nbands = std::min<u64>(nbands, (u64)cam.tiles_y);
    const int band_rows = (int)(((u64)cam.tiles_y + nbands - 1) / nbands);
    const int nb = (cam.tiles_y + band_rows - 1) / band_rows;
    const size_t smem_place = 2 * (size_t)band_rows * cam.tiles_x * sizeof(u32);
    if (smem_place > 48 * 1024)
      cudaFuncSetAttribute(tile_place_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_place);
    launch_pdl(tile_place_kernel<256>, dim3(kChunks, nb), 256, smem_place, st, ntiles, cam.tiles_x, ws.recs, ws.bounds,
               ws.chunk_table, ranges, bin.num_instances, bin.capacity, band_rows, bin.ids);
    launched();
    if (bin.keys) {
      launch_pdl(tile_keys_kernel, (ntiles + 1) / 2, 256, 0, st, ntiles, (const uint2*)ranges, (const u32*)bin.ids, proj.depth, bin.keys);
      launched();
    }
    tm.end(st);
    return cudaGetLastError();
  }
  // images with more tiles than the counting pass can histogram in shared memory: one-byte LSD passes on the
  // tile id over the duplicated instances
  unsigned long long* total64 = reinterpret_cast<unsigned long long*>(ws.count_a);
  cudaMemsetAsync(total64, 0, sizeof(unsigned long long), st);
  instance_total_kernel<<<sm_count() * 4, 256, 0, st>>>(N, proj.tiles_touched, total64);
  clamp_count_kernel<<<1, 1, 0, st>>>(ws.count_b, bin.num_instances, total64, bin.capacity);
  launched(2);
  // stage B passes: one per byte of the tile id.  The last pass reads the alternate buffers and writes
  // bin.keys / bin.ids; earlier passes ping-pong between (bin.keys viewed as u32, bin.ids) and the alternates.
  int tile_bits = 0;
  while ((1 << tile_bits) < ntiles) ++tile_bits;
  const int passes = tile_bits <= 8 ? 1 : (tile_bits + 7) / 8;
  u32* kbuf[2] = {reinterpret_cast<u32*>(bin.keys), ws.ik};  // [1] = alternates
  u32* vbuf[2] = {bin.ids, ws.iv};
  int cur = (passes & 1) ? 1 : 0;  // input of pass 0, chosen so that the last pass reads the alternates
  // K3
  tm.begin(GABSPLAT_STAGE_DUPLICATE, st);
  duplicate_kernel<<<(u32)((bin.capacity + kDupChunk - 1) / kDupChunk), kDupThreads, 0, st>>>(
      ws.n_vis, cam.tiles_x, order, bin.offsets, reinterpret_cast<const int4*>(proj.rect), bin.num_instances, bin.capacity,
      kbuf[cur], vbuf[cur]);
  launched();
  tm.end(st);
  // B
  tm.begin(GABSPLAT_STAGE_SORT, st);
  const u32 nbb = sort_blocks(bin.capacity);
  for (int p = 0; p < passes; ++p) {
    const bool final_pass = p == passes - 1;
    radix_pass(kbuf[cur], vbuf[cur], kbuf[cur ^ 1], vbuf[cur ^ 1], final_pass ? bin.keys : nullptr,
               reinterpret_cast<const u32*>(proj.depth), ws.count_b, nbb, 8 * p, ws, st);
    cur ^= 1;
  }
  tm.end(st);
  // K5
  tm.begin(GABSPLAT_STAGE_RANGES, st);
  cudaMemsetAsync(bin.tile_ranges, 0, (size_t)ntiles * 2 * sizeof(u32), st);
  tile_ranges_kernel<<<sm_count() * 8, 256, 0, st>>>(bin.keys, bin.num_instances, bin.capacity,
                                              reinterpret_cast<uint2*>(bin.tile_ranges));
  launched();
  const cudaError_t eo = launch_tile_order(bin.tile_ranges, false, ntiles, bin.tile_order, st);
  tm.end(st);
  return eo != cudaSuccess ? eo : cudaGetLastError();
}

}  // namespace gabsplat
