// Exclusive prefix scan of uint32 arrays of arbitrary length (three launches: tile sums, scan of the tile sums,
// rescan with carry-in).  Used for the grid's bin offsets ("prefix scan" of BASELINE.json L5 item 1), the
// start-hit compaction and the track / track-hit offsets.  HBM traffic: 2 reads + 1 write of the array.
#pragma once
#include "common.cuh"

namespace tpc {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;   // 4096 elements per CTA

__device__ __forceinline__ uint32_t warp_inclusive_scan(uint32_t v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, v, d);
    if (lane_id() >= (unsigned)d) v += t;
  }
  return v;
}

// Exclusive scan of one value per thread across a CTA of kScanThreads threads; returns the CTA total in `total`.
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t& total) {
  __shared__ uint32_t warp_sums[kScanThreads / 32];
  const uint32_t inc = warp_inclusive_scan(v);
  const int w = threadIdx.x >> 5;
  if (lane_id() == 31) warp_sums[w] = inc;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (int i = 0; i < kScanThreads / 32; ++i) {
    const uint32_t s = warp_sums[i];
    if (i < w) base += s;
    tot += s;
  }
  __syncthreads();
  total = tot;
  return base + inc - v;
}

// Pass 1: tile_sums[b] = sum of tile b.  Each thread owns kScanItems consecutive elements (vector-friendly).
__global__ void __launch_bounds__(kScanThreads) k_scan_tile_sums(const uint32_t* __restrict__ in, uint32_t* __restrict__ tile_sums, size_t n) {
  const size_t base = (size_t)blockIdx.x * kScanTile + (size_t)threadIdx.x * kScanItems;
  uint32_t s = 0;
  if (base + kScanItems <= n && (reinterpret_cast<uintptr_t>(in) & 15) == 0) {
    const uint4* p = reinterpret_cast<const uint4*>(in + base);
#pragma unroll
    for (int i = 0; i < kScanItems / 4; ++i) { const uint4 v = p[i]; s += v.x + v.y + v.z + v.w; }
  } else {
    for (int i = 0; i < kScanItems; ++i) if (base + i < n) s += in[base + i];
  }
  uint32_t total;
  block_exclusive_scan(s, total);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

// Pass 2 (one CTA): exclusive scan of the tile sums in place; tile_sums[n_tiles] = grand total.
__global__ void __launch_bounds__(kScanThreads) k_scan_tile_offsets(uint32_t* __restrict__ tile_sums, int n_tiles) {
  uint32_t carry = 0;
  for (int base = 0; base < n_tiles; base += kScanThreads) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < n_tiles ? tile_sums[i] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(v, total);
    if (i < n_tiles) tile_sums[i] = carry + ex;
    carry += total;
  }
  if (threadIdx.x == 0) tile_sums[n_tiles] = carry;
}

// Pass 3: out[i] = tile offset + exclusive scan inside the tile.  in == out is allowed.
// If total_out != nullptr the grand total is also written there as int32 / int64 (device scalars).
__global__ void __launch_bounds__(kScanThreads) k_scan_apply(const uint32_t* in, uint32_t* out, const uint32_t* __restrict__ tile_sums, size_t n) {
  const size_t base = (size_t)blockIdx.x * kScanTile + (size_t)threadIdx.x * kScanItems;
  uint32_t v[kScanItems];
  const bool vec = base + kScanItems <= n && (reinterpret_cast<uintptr_t>(in) & 15) == 0 && (reinterpret_cast<uintptr_t>(out) & 15) == 0;
  if (vec) {
    const uint4* p = reinterpret_cast<const uint4*>(in + base);
#pragma unroll
    for (int i = 0; i < kScanItems / 4; ++i) { const uint4 q = p[i]; v[4 * i] = q.x; v[4 * i + 1] = q.y; v[4 * i + 2] = q.z; v[4 * i + 3] = q.w; }
  } else {
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) v[i] = base + i < n ? in[base + i] : 0u;
  }
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) s += v[i];
  uint32_t total;
  uint32_t run = block_exclusive_scan(s, total) + tile_sums[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) { const uint32_t t = v[i]; v[i] = run; run += t; }
  if (vec) {
    uint4* p = reinterpret_cast<uint4*>(out + base);
#pragma unroll
    for (int i = 0; i < kScanItems / 4; ++i) p[i] = make_uint4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
  } else {
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) if (base + i < n) out[base + i] = v[i];
  }
}

// Host helper: exclusive scan of in[0..n) into out[0..n) (in == out allowed).  `tile_sums` needs
// ceil(n / kScanTile) + 1 entries; afterwards tile_sums[n_tiles] holds the grand total.  Returns launches.
inline int exclusive_scan_u32(const uint32_t* in, uint32_t* out, size_t n, uint32_t* tile_sums, cudaStream_t st) {
  if (n == 0) return 0;
  const int n_tiles = (int)((n + kScanTile - 1) / kScanTile);
  k_scan_tile_sums<<<n_tiles, kScanThreads, 0, st>>>(in, tile_sums, n);
  k_scan_tile_offsets<<<1, kScanThreads, 0, st>>>(tile_sums, n_tiles);
  k_scan_apply<<<n_tiles, kScanThreads, 0, st>>>(in, out, tile_sums, n);
  return 3;
}
inline size_t scan_tiles(size_t n) { return (n + kScanTile - 1) / kScanTile; }

}  // namespace tpc
