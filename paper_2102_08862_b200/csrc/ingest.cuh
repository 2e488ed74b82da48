// C1 cluster ingest (BASELINE.json L5 item 1: "sorts clusters into per-(sector, row) grids of (pad, time) bins by
// radix sort and prefix scan"; PAPER.md L23 native coordinates).
//
// key(i) = ((sector*n_rows + row) * n_tb + time_bin(time)) * n_pb + pad_bin(y)   (= grid bin index, common.cuh::grid_bin;
// n_bins for clusters outside the geometry, which therefore sort to the end).  A stable least-significant-digit radix sort
// on the key orders the frame by (sector-row, time bin, pad bin) and, inside a bin, by original index -- the layout is
// deterministic.
// One pass = k_radix_histogram (digit counts per 2048-element tile) -> exclusive prefix scan over
// (digit, tile) -> k_radix_scatter (stable in-tile ranking by warp match, local reorder in shared memory, then
// every digit's run is written contiguously: coalesced writes instead of 4..8-byte random scatters).
// The first pass reads the raw fp32 SoA input and converts pad -> local y on the fly; the last pass writes the
// final hit arrays.  k_grid_build then derives the grid's bin offsets from the sorted keys (no atomics).
//
// Algorithmic HBM bytes per cluster: passes * (4 + 16 + 16) + grid build ~ 8.
#pragma once
#include "common.cuh"

namespace tpc {

#ifndef TPC_RADIX_THREADS
#define TPC_RADIX_THREADS 256
#endif
constexpr int kRadixThreads = TPC_RADIX_THREADS;
constexpr int kRadixItems = 8;
constexpr int kRadixTile = kRadixThreads * kRadixItems;   // 2048 (256 threads) or 4096 (512)
constexpr int kRadixMaxBits = 8;
constexpr int kRadixBuckets = 1 << kRadixMaxBits;
constexpr size_t kRadixScatterSmem = (size_t)kRadixTile * 16 + (size_t)(kRadixThreads / 32 + 2) * kRadixBuckets * 4;

// A cluster is inside the geometry iff row is an integer in [0, n_sr), pad in [-0.5, n_pads-0.5) and
// time in [0, max_time]; evaluated in fp32 on the raw values (DESIGN.md §3 C1).
// Also returns the local y of a valid cluster.
__device__ __forceinline__ uint32_t cluster_key(float rf, float pad, float time, const Consts& c, float& y) {
  const bool ok_row = rf >= 0.0f && rf < (float)c.n_sr && rf == floorf(rf);
  const int sr = ok_row ? (int)rf : 0;
  // r = sr mod n_rows without an integer division: sr < 2^16 and n_rows <= 160, so (sr + 0.5) / n_rows is at least
  // 0.003 away from an integer while the fp32 product is off by < 1e-4
  const int r = sr - (int)(((float)sr + 0.5f) * c.inv_n_rows) * c.n_rows;
  const float4 rt = __ldg(c.rowtab + r);                                // (n_pads - 0.5 [exact in fp32], c_r, yoff, pscale)
  const bool ok = ok_row && pad >= -0.5f && pad < rt.x && time >= 0.0f && time <= c.max_time;
  y = ok ? (pad - rt.y) * c.P : 0.0f;                                   // y(h) = (pad - c_r) * P
  const uint32_t key = grid_bin(sr, time_bin(time, c), pad_bin(y, rt.z, rt.w, c), c);
  return ok ? key : (uint32_t)c.n_bins;
}

struct RadixSrc {        // input of a pass: either the raw clusters (first pass) or a sorted-so-far set
  const float* row; const float* pad; const float* time;        // first pass
  const uint32_t* keys; const uint32_t* orig; const float2* yt; // later passes
};
struct RadixDst { uint32_t* keys; uint32_t* orig; float2* yt; };

// Digit histogram of one tile: hist[digit * n_tiles + tile].
template <bool kFirst>
__global__ void __launch_bounds__(kRadixThreads) k_radix_histogram(RadixSrc src, int64_t n, int shift, uint32_t mask,
                                                                   uint32_t* __restrict__ hist, int n_tiles,
                                                                   const __grid_constant__ Consts c) {
  __shared__ uint32_t cnt[kRadixBuckets];
  for (int i = threadIdx.x; i < kRadixBuckets; i += kRadixThreads) cnt[i] = 0;
  __syncthreads();
  const int64_t base = (int64_t)blockIdx.x * kRadixTile;
  if (kFirst) {                                     // all loads of the tile first, then the key arithmetic
    float rf[kRadixItems], pd[kRadixItems], tm[kRadixItems];
#pragma unroll
    for (int k = 0; k < kRadixItems; ++k) {
      const int64_t i = base + (int64_t)k * kRadixThreads + threadIdx.x;
      const bool in = i < n;
      rf[k] = in ? src.row[i] : -1.0f; pd[k] = in ? src.pad[i] : 0.0f; tm[k] = in ? src.time[i] : 0.0f;
    }
#pragma unroll
    for (int k = 0; k < kRadixItems; ++k) {
      float y;
      const uint32_t key = cluster_key(rf[k], pd[k], tm[k], c, y);
      if (base + (int64_t)k * kRadixThreads + threadIdx.x < n) atomicAdd(&cnt[(key >> shift) & mask], 1u);
    }
  } else {
#pragma unroll
    for (int k = 0; k < kRadixItems; ++k) {
      const int64_t i = base + (int64_t)k * kRadixThreads + threadIdx.x;
      if (i < n) atomicAdd(&cnt[(src.keys[i] >> shift) & mask], 1u);
    }
  }
  __syncthreads();
  for (int d = threadIdx.x; d <= (int)mask; d += kRadixThreads) hist[(size_t)d * n_tiles + blockIdx.x] = cnt[d];
}

// Stable scatter of one tile.  `offsets` = exclusive scan of hist (same layout): global position of the first
// element of (digit, tile).
#ifndef TPC_SCATTER_CTAS
#define TPC_SCATTER_CTAS 4
#endif
template <bool kFirst>
__global__ void __launch_bounds__(kRadixThreads, TPC_SCATTER_CTAS) k_radix_scatter(RadixSrc src, RadixDst dst, int64_t n, int shift, uint32_t mask,
                                                                 const uint32_t* __restrict__ offsets, int n_tiles,
                                                                 uint32_t* __restrict__ n_invalid,
                                                                 const __grid_constant__ Consts c) {
  constexpr int kWarps = kRadixThreads / 32;
  constexpr int kWarpItems = kRadixTile / kWarps;                 // 256 consecutive elements per warp
  extern __shared__ __align__(16) unsigned char radix_smem[];     // kRadixScatterSmem bytes (dynamic: > 48 KB)
  float2* s_yt = reinterpret_cast<float2*>(radix_smem);                                   // [kRadixTile]
  uint32_t* s_keys = reinterpret_cast<uint32_t*>(s_yt + kRadixTile);                      // [kRadixTile]
  uint32_t* s_orig = s_keys + kRadixTile;                                                 // [kRadixTile]
  uint32_t (*warp_cnt)[kRadixBuckets] = reinterpret_cast<uint32_t (*)[kRadixBuckets]>(s_orig + kRadixTile);  // per-warp digit counts
  uint32_t* digit_start = &warp_cnt[kWarps][0];                   // first local position of each digit in the tile
  uint32_t* gbase = digit_start + kRadixBuckets;                  // global position of the tile's first element of a digit
  const int w = threadIdx.x >> 5;
  const unsigned lane = lane_id();
  const int n_dig = (int)mask + 1;
  for (int i = threadIdx.x; i < kWarps * kRadixBuckets; i += kRadixThreads) (&warp_cnt[0][0])[i] = 0;
  __syncthreads();

  // 1. load (warp w owns elements [w*256, w*256+256) of the tile, lane-strided -> coalesced)
  const int64_t tile_base = (int64_t)blockIdx.x * kRadixTile;
  const int64_t wbase = tile_base + (int64_t)w * kWarpItems;
  uint32_t key[kRadixItems], og[kRadixItems], rank[kRadixItems];
  float2 yt[kRadixItems];
  const int n_mine = (int)min((int64_t)kWarpItems, max(n - wbase, (int64_t)0));   // elements of this warp's slice that exist
  if (kFirst) {
    float rf[kRadixItems];
#pragma unroll
    for (int k = 0; k < kRadixItems; ++k) {           // all loads first, then the key arithmetic
      const bool in = k * 32 + (int)lane < n_mine;
      const int64_t i = wbase + k * 32 + lane;
      rf[k] = in ? src.row[i] : -1.0f; yt[k].x = in ? src.pad[i] : 0.0f; yt[k].y = in ? src.time[i] : 0.0f;
      og[k] = (uint32_t)i;
    }
    uint32_t bad = 0;
#pragma unroll
    for (int k = 0; k < kRadixItems; ++k) {
      float y;
      key[k] = cluster_key(rf[k], yt[k].x, yt[k].y, c, y);
      yt[k].x = y;
      if (k * 32 + (int)lane < n_mine && key[k] == (uint32_t)c.n_bins) ++bad;
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    if (bad && lane == 0) atomicAdd(n_invalid, bad);
  } else {
#pragma unroll
    for (int k = 0; k < kRadixItems; ++k) {
      const bool in = k * 32 + (int)lane < n_mine;
      const int64_t i = wbase + k * 32 + lane;
      key[k] = in ? src.keys[i] : 0xFFFFFFFFu; og[k] = in ? src.orig[i] : 0u; yt[k] = in ? src.yt[i] : make_float2(0.0f, 0.0f);
    }
  }

  // 2. stable rank inside the warp: elements are visited in index order (k-major, lane-minor).  The eight warp
  // matches are independent and issued back to back; only the counter updates form a chain.
  unsigned peers[kRadixItems];
#pragma unroll
  for (int k = 0; k < kRadixItems; ++k) {
    const bool valid = k * 32 + (int)lane < n_mine;
    const uint32_t d = valid ? (key[k] >> shift) & mask : mask + 1u;      // padding never matches a digit
    peers[k] = __match_any_sync(0xffffffffu, d);
  }
#pragma unroll
  for (int k = 0; k < kRadixItems; ++k) {
    const bool valid = k * 32 + (int)lane < n_mine;
    const uint32_t d = (key[k] >> shift) & mask;
    const int leader = __ffs(peers[k]) - 1;
    uint32_t before = 0;
    if (valid && (int)lane == leader) { before = warp_cnt[w][d]; warp_cnt[w][d] = before + __popc(peers[k]); }
    before = __shfl_sync(0xffffffffu, before, leader);
    rank[k] = before + __popc(peers[k] & ((1u << lane) - 1u));
    __syncwarp();
  }
  __syncthreads();

  // 3. per digit: exclusive offsets over the warps, tile totals, then an exclusive scan over the digits
  uint32_t tile_total = 0;
  if ((int)threadIdx.x < n_dig) {
    uint32_t run = 0;
#pragma unroll
    for (int ww = 0; ww < kWarps; ++ww) { const uint32_t t = warp_cnt[ww][threadIdx.x]; warp_cnt[ww][threadIdx.x] = run; run += t; }
    tile_total = run;
    gbase[threadIdx.x] = offsets[(size_t)threadIdx.x * n_tiles + blockIdx.x];
  }
  {
    // block exclusive scan of tile_total over threads 0..255 (n_dig <= 256)
    __shared__ uint32_t wsum[kWarps];
    uint32_t inc = tile_total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o); if ((int)lane >= o) inc += t; }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    uint32_t pre = 0;
    for (int ww = 0; ww < w; ++ww) pre += wsum[ww];
    if ((int)threadIdx.x < n_dig) digit_start[threadIdx.x] = pre + inc - tile_total;
  }
  __syncthreads();

  // 4. local reorder into shared memory
#pragma unroll
  for (int k = 0; k < kRadixItems; ++k) {
    if (k * 32 + (int)lane < n_mine) {
      const uint32_t d = (key[k] >> shift) & mask;
      const uint32_t pos = digit_start[d] + warp_cnt[w][d] + rank[k];
      s_keys[pos] = key[k]; s_orig[pos] = og[k]; s_yt[pos] = yt[k];
    }
  }
  __syncthreads();

  // 5. write every digit's run contiguously
  const int n_here = (int)min((int64_t)kRadixTile, n - tile_base);
  for (int p = threadIdx.x; p < n_here; p += kRadixThreads) {
    const uint32_t kk = s_keys[p];
    const uint32_t d = (kk >> shift) & mask;
    const uint32_t g = gbase[d] + ((uint32_t)p - digit_start[d]);
    dst.keys[g] = kk; dst.orig[g] = s_orig[p]; dst.yt[g] = s_yt[p];
  }
}

// Grid bin offsets from the sorted keys: bin_start[b] = first position whose key >= b, for b in [0, n_bins].
// Thread i (0 <= i <= n) fills the bins in (key[i-1], key[i]]; also writes the hit's sector-row (u16).  On a dense frame a
// gap is one or two bins.  A gap longer than kGridGapInline (an empty or sparse frame on a long-frame grid: up to all 2.8e8
// bins) is not written by the one thread but cut into segments of kGridGapSegment bins that k_grid_fill_gaps fills with a
// CTA each -- no thread ever writes more than kGridGapInline entries one by one.
constexpr int kGridGapInline = 64, kGridGapSegment = 4096;
__global__ void __launch_bounds__(256) k_grid_build(const uint32_t* __restrict__ keys, int64_t n, uint32_t* __restrict__ bin_start,
                                                    uint16_t* __restrict__ hsr, uint4* __restrict__ gap_list, uint32_t* __restrict__ n_gaps,
                                                    const __grid_constant__ Consts c) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i > n) return;
  const uint32_t nb = (uint32_t)c.n_bins;
  const int64_t kprev = i == 0 ? -1 : (int64_t)min(keys[i - 1], nb);
  const uint32_t kcur = i == n ? nb : min(keys[i], nb);
  if (i < n && kcur < nb) hsr[i] = (uint16_t)(kcur / (uint32_t)(c.n_tb * c.n_pb));
  const int64_t len = (int64_t)kcur - kprev;
  if (len <= kGridGapInline) {
    for (int64_t b = kprev + 1; b <= (int64_t)kcur; ++b) bin_start[b] = (uint32_t)i;
  } else {
    const uint32_t n_seg = (uint32_t)((len + kGridGapSegment - 1) / kGridGapSegment);
    const uint32_t base = atomicAdd(n_gaps, n_seg);
    for (uint32_t s = 0; s < n_seg; ++s) {
      const int64_t b0 = kprev + 1 + (int64_t)s * kGridGapSegment;
      gap_list[base + s] = make_uint4((uint32_t)b0, (uint32_t)min(b0 + kGridGapSegment, (int64_t)kcur + 1), (uint32_t)i, 0u);
    }
  }
}
// bin_start[b0 .. b1) = value for every listed segment (any order: the segments are disjoint)
__global__ void __launch_bounds__(256) k_grid_fill_gaps(const uint4* __restrict__ gap_list, const uint32_t* __restrict__ n_gaps,
                                                        uint32_t* __restrict__ bin_start) {
  const uint32_t n = *n_gaps;
  for (uint32_t s = blockIdx.x; s < n; s += gridDim.x) {
    const uint4 g = gap_list[s];
    for (uint32_t b = g.x + threadIdx.x; b < g.y; b += blockDim.x) bin_start[b] = g.z;
  }
}

}  // namespace tpc
