// S2 / K2-K5: tile binning.  (PAPER.md:103 "sorted by depth", :160 "tile-based rasterizer".)
//   K2  inclusive prefix sum of tiles_touched                       -> offsets, D
//   K3  one (key,id) per (primitive, tile of its rectangle), primitive-major, row-major over the rectangle,
//       key = (tile << 32) | bits(depth)
//   K4  stable LSD radix sort of the pairs on one-byte digits (in-house; no library sort)
//   K5  [start,end) of every tile in the sorted list
// Everything is integer work; the result must equal std::stable_sort of the keys bit for bit.
// The instance count D lives on the device: every kernel is launched on a grid sized from the caller's
// capacity and returns early past D, so the whole stage runs without a host round trip.
#include "common.cuh"

namespace gabsplat {
namespace {

typedef uint32_t u32;
typedef uint64_t u64;

// ------------------------------------------------------------------------------------------------
// Device-wide prefix sum of u32 (three launches: block sums, scan of the sums, block scans).
// ------------------------------------------------------------------------------------------------
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

__global__ void __launch_bounds__(kScanThreads) scan_block_sums(const u32* __restrict__ in, u32 n, u32* __restrict__ sums) {
  const u32 base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  u32 s = 0;
  if (base + kScanItems <= n) {
    const uint4* p = reinterpret_cast<const uint4*>(in + base);
#pragma unroll
    for (int j = 0; j < kScanItems / 4; ++j) { const uint4 v = p[j]; s += v.x + v.y + v.z + v.w; }
  } else {
    for (int j = 0; j < kScanItems; ++j) if (base + j < n) s += in[base + j];
  }
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

template <bool INCLUSIVE>
__global__ void __launch_bounds__(kScanThreads) scan_apply(const u32* __restrict__ in, u32 n, const u32* __restrict__ sums,
                                                            u32* __restrict__ out) {
  const u32 base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  u32 v[kScanItems];
  const bool full = base + kScanItems <= n;
  if (full) {
    const uint4* p = reinterpret_cast<const uint4*>(in + base);
#pragma unroll
    for (int j = 0; j < kScanItems / 4; ++j) {
      const uint4 x = p[j];
      v[4 * j] = x.x; v[4 * j + 1] = x.y; v[4 * j + 2] = x.z; v[4 * j + 3] = x.w;
    }
  } else {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) v[j] = base + j < n ? in[base + j] : 0;
  }
  u32 s = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) s += v[j];
  u32 total;
  u32 run = block_exclusive_scan(s, &total) + sums[blockIdx.x];
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    const u32 e = run;
    run += v[j];
    v[j] = INCLUSIVE ? run : e;
  }
  if (full) {
    uint4* q = reinterpret_cast<uint4*>(out + base);
#pragma unroll
    for (int j = 0; j < kScanItems / 4; ++j) q[j] = make_uint4(v[4 * j], v[4 * j + 1], v[4 * j + 2], v[4 * j + 3]);
  } else {
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) if (base + j < n) out[base + j] = v[j];
  }
}

inline u32 scan_blocks(u32 n) { return (n + kScanTile - 1) / kScanTile; }

// sums must hold scan_blocks(n) u32.  in/out must be 16-byte aligned.  in == out is allowed.
template <bool INCLUSIVE>
void device_scan(const u32* in, u32* out, u32 n, u32* sums, u32* total_out, cudaStream_t st) {
  const u32 nb = scan_blocks(n);
  if (nb == 0) {
    scan_of_sums<<<1, kScanThreads, 0, st>>>(sums, 0, total_out);
    launched();
    return;
  }
  scan_block_sums<<<nb, kScanThreads, 0, st>>>(in, n, sums);
  launched();
  scan_of_sums<<<1, kScanThreads, 0, st>>>(sums, nb, total_out);
  launched();
  scan_apply<INCLUSIVE><<<nb, kScanThreads, 0, st>>>(in, n, sums, out);
  launched();
}

// ------------------------------------------------------------------------------------------------
// K3: duplicate.  One block per 256 primitives; the block's instances are emitted cooperatively so that
// writes are coalesced and a primitive covering thousands of tiles is shared by the whole block.
// ------------------------------------------------------------------------------------------------
constexpr int kDupThreads = 256;

__global__ void __launch_bounds__(kDupThreads) duplicate_kernel(int N, int tiles_x, const u32* __restrict__ offsets,
                                                               const u32* __restrict__ tiles_touched,
                                                               const int4* __restrict__ rect, const float* __restrict__ depth,
                                                               const u32* __restrict__ num_instances, u64 capacity,
                                                               u64* __restrict__ keys, u32* __restrict__ ids) {
  __shared__ u32 s_incl[kDupThreads];
  __shared__ int4 s_rect[kDupThreads];
  __shared__ u32 s_depth[kDupThreads];
  if ((u64)*num_instances > capacity) return;
  const int i0 = blockIdx.x * kDupThreads;
  const int i = i0 + threadIdx.x;
  u32 incl = 0, tt = 0;
  if (i < N) { incl = offsets[i]; tt = tiles_touched[i]; }
  else if (N > 0) incl = offsets[N - 1];
  s_incl[threadIdx.x] = incl;
  if (tt) { s_rect[threadIdx.x] = rect[i]; s_depth[threadIdx.x] = __float_as_uint(depth[i]); }
  __shared__ u32 s_base;
  if (threadIdx.x == 0) s_base = incl - tt;
  __syncthreads();
  const u32 base = s_base;
  const u32 count = s_incl[kDupThreads - 1] - base;
  for (u32 e = threadIdx.x; e < count; e += kDupThreads) {
    const u32 g = base + e;
    // first p with s_incl[p] > g
    int lo = 0, hi = kDupThreads - 1;
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if (s_incl[mid] > g) hi = mid; else lo = mid + 1;
    }
    const int4 r = s_rect[lo];
    const u32 first = lo ? s_incl[lo - 1] : base;
    const u32 local = g - first;
    const u32 w = (u32)(r.z - r.x);
    const u32 row = local / w, col = local - row * w;
    const u32 tile = (u32)(r.y + row) * (u32)tiles_x + (u32)r.x + col;
    keys[g] = ((u64)tile << 32) | (u64)s_depth[lo];
    ids[g] = (u32)(i0 + lo);
  }
}

// ------------------------------------------------------------------------------------------------
// K4: one LSD radix pass on the one-byte digit (key >> shift) & 255: per-block digit histogram,
// scan of the [digit][block] table, stable scatter.
// ------------------------------------------------------------------------------------------------
constexpr int kSortThreads = 256;
constexpr int kSortItems = 8;
constexpr int kSortTile = kSortThreads * kSortItems;  // 2048 pairs per block
constexpr int kSortWarps = kSortThreads / 32;

__global__ void __launch_bounds__(kSortThreads) sort_histogram(const u64* __restrict__ keys, const u32* __restrict__ num_instances,
                                                              u32* __restrict__ table, u32 nblocks, int shift) {
  __shared__ u32 hist[256];
  hist[threadIdx.x] = 0;
  __syncthreads();
  const u32 D = *num_instances;
  const u32 start = blockIdx.x * kSortTile;
  if (start < D) {
    const u32 n = min((u32)kSortTile, D - start);
    for (u32 j = threadIdx.x; j < n; j += kSortThreads) atomicAdd(&hist[(u32)(keys[start + j] >> shift) & 255u], 1u);
  }
  __syncthreads();
  table[threadIdx.x * nblocks + blockIdx.x] = hist[threadIdx.x];
}

__global__ void __launch_bounds__(kSortThreads) sort_scatter(const u64* __restrict__ kin, const u32* __restrict__ vin,
                                                            u64* __restrict__ kout, u32* __restrict__ vout,
                                                            const u32* __restrict__ num_instances,
                                                            const u32* __restrict__ table, u32 nblocks, int shift) {
  __shared__ u32 warp_hist[kSortWarps][256];
  __shared__ u32 local_base[256];
  __shared__ u32 global_base[256];
  __shared__ u64 skeys[kSortTile];
  __shared__ u32 svals[kSortTile];
  const u32 D = *num_instances;
  const u32 start = blockIdx.x * kSortTile;
  if (start >= D) return;
  const u32 n = min((u32)kSortTile, D - start);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int j = 0; j < kSortWarps; ++j) warp_hist[j][threadIdx.x] = 0;
  __syncthreads();

  u64 k[kSortItems];
  u32 v[kSortItems], rank[kSortItems];
  const u32 lt_mask = (1u << lane) - 1u;
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const u32 idx = (u32)w * 32u * kSortItems + (u32)r * 32u + (u32)lane;
    const bool valid = idx < n;
    k[r] = valid ? kin[start + idx] : 0;
    v[r] = valid ? vin[start + idx] : 0;
    const u32 d = (u32)(k[r] >> shift) & 255u;
    // lanes holding the same digit (valid lanes only)
    u32 peers = __ballot_sync(0xffffffffu, valid);
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      const u32 bal = __ballot_sync(0xffffffffu, (d >> b) & 1u);
      peers &= ((d >> b) & 1u) ? bal : ~bal;
    }
    u32 prev = 0;
    const int leader = __ffs(peers) - 1;
    if (valid && lane == leader) {
      prev = warp_hist[w][d];
      warp_hist[w][d] = prev + __popc(peers);
    }
    prev = __shfl_sync(0xffffffffu, prev, valid ? leader : lane);
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
    global_base[d] = table[(u32)d * nblocks + blockIdx.x];
  }
  __syncthreads();
#pragma unroll
  for (int r = 0; r < kSortItems; ++r) {
    const u32 idx = (u32)w * 32u * kSortItems + (u32)r * 32u + (u32)lane;
    if (idx < n) {
      const u32 d = (u32)(k[r] >> shift) & 255u;
      const u32 pos = local_base[d] + warp_hist[w][d] + rank[r];
      skeys[pos] = k[r];
      svals[pos] = v[r];
    }
  }
  __syncthreads();
  for (u32 j = threadIdx.x; j < n; j += kSortThreads) {
    const u64 key = skeys[j];
    const u32 d = (u32)(key >> shift) & 255u;
    const u32 dst = global_base[d] + (j - local_base[d]);
    kout[dst] = key;
    vout[dst] = svals[j];
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

__global__ void clamp_count_kernel(u32* sort_count, const u32* num_instances, u64 capacity) {
  // the sort kernels see 0 instances when the caller's buffers are too small
  *sort_count = (u64)*num_instances > capacity ? 0u : *num_instances;
}

inline u64 align_up(u64 x, u64 a) { return (x + a - 1) / a * a; }

struct Workspace {
  u32* scan_sums;   // scan partials (reused by every scan)
  u32* sort_count;  // [1]
  u32* table;       // [256][nblocks]
  u64* keys_alt;
  u32* ids_alt;
  u64 bytes;
};

Workspace carve(void* base, int N, u64 capacity) {
  const u32 nblocks = (u32)((capacity + kSortTile - 1) / kSortTile);
  const u64 table_n = (u64)256 * (nblocks ? nblocks : 1);
  const u64 sums_n = (u64)scan_blocks((u32)(table_n > (u64)N ? table_n : (u64)N)) + 16;
  u64 off = 0;
  Workspace w;
  char* b = (char*)base;
  w.scan_sums = (u32*)(b + off); off = align_up(off + sums_n * 4, 256);
  w.sort_count = (u32*)(b + off); off = align_up(off + 16, 256);
  w.table = (u32*)(b + off); off = align_up(off + table_n * 4, 256);
  w.keys_alt = (u64*)(b + off); off = align_up(off + capacity * 8, 256);
  w.ids_alt = (u32*)(b + off); off = align_up(off + capacity * 4, 256);
  w.bytes = off;
  return w;
}

}  // namespace

uint64_t sort_workspace_bytes(int N, uint64_t capacity) { return carve(nullptr, N, capacity).bytes; }

cudaError_t launch_bin_sort(int N, const gabsplat_projected& proj, const Camera& cam, const gabsplat_binning& bin,
                            StageTimer& tm, cudaStream_t st) {
  const Workspace ws = carve(bin.workspace, N, bin.capacity);
  const int ntiles = cam.tiles_x * cam.tiles_y;
  // K2
  tm.begin(GABSPLAT_STAGE_SCAN, st);
  device_scan<true>(proj.tiles_touched, bin.offsets, (u32)N, ws.scan_sums, bin.num_instances, st);
  tm.end(st);
  if (N == 0 || bin.capacity == 0) {
    cudaMemsetAsync(bin.tile_ranges, 0, (size_t)ntiles * 2 * sizeof(u32), st);
    return cudaGetLastError();
  }
  clamp_count_kernel<<<1, 1, 0, st>>>(ws.sort_count, bin.num_instances, bin.capacity);
  launched();
  // number of one-byte passes: 32 depth bits + bits of the largest tile id
  int tile_bits = 0;
  while ((1 << tile_bits) < ntiles) ++tile_bits;
  const int passes = (32 + tile_bits + 7) / 8;
  u64* kbuf[2] = {bin.keys, ws.keys_alt};
  u32* vbuf[2] = {bin.ids, ws.ids_alt};
  int cur = passes & 1;  // an odd number of passes starts in the alternate buffer so the result lands in bin.keys
  // K3
  tm.begin(GABSPLAT_STAGE_DUPLICATE, st);
  duplicate_kernel<<<(N + kDupThreads - 1) / kDupThreads, kDupThreads, 0, st>>>(
      N, cam.tiles_x, bin.offsets, proj.tiles_touched, reinterpret_cast<const int4*>(proj.rect), proj.depth,
      bin.num_instances, bin.capacity, kbuf[cur], vbuf[cur]);
  launched();
  tm.end(st);
  // K4
  tm.begin(GABSPLAT_STAGE_SORT, st);
  const u32 nblocks = (u32)((bin.capacity + kSortTile - 1) / kSortTile);
  for (int p = 0; p < passes; ++p) {
    const int shift = 8 * p;
    sort_histogram<<<nblocks, kSortThreads, 0, st>>>(kbuf[cur], ws.sort_count, ws.table, nblocks, shift);
    launched();
    device_scan<false>(ws.table, ws.table, 256u * nblocks, ws.scan_sums, nullptr, st);
    sort_scatter<<<nblocks, kSortThreads, 0, st>>>(kbuf[cur], vbuf[cur], kbuf[cur ^ 1], vbuf[cur ^ 1], ws.sort_count,
                                                   ws.table, nblocks, shift);
    launched();
    cur ^= 1;
  }
  tm.end(st);
  // K5
  tm.begin(GABSPLAT_STAGE_RANGES, st);
  cudaMemsetAsync(bin.tile_ranges, 0, (size_t)ntiles * 2 * sizeof(u32), st);
  tile_ranges_kernel<<<148 * 8, 256, 0, st>>>(bin.keys, bin.num_instances, bin.capacity,
                                              reinterpret_cast<uint2*>(bin.tile_ranges));
  launched();
  tm.end(st);
  return cudaGetLastError();
}

}  // namespace gabsplat
