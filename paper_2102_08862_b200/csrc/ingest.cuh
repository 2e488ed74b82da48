// C1 cluster ingest (BASELINE.json L5 item 1; PAPER.md L23 native coordinates): sorts the frame's clusters
// into per-(sector,row) grids of time bins -- a one-digit radix (counting) sort on the key
// (sector*n_rows + row, time_bin) with a prefix scan of the bin histogram -- and converts pad -> local y.
//
//   k_ingest_count  : validity, key, rank[i] = atomicAdd(binCount[key], 1)             (12 B read, 4 B write)
//   exclusive scan  : binStart = scan(binCount)                                        (scan.cuh)
//   k_ingest_scatter: pos = binStart[key] + rank[i]; yt[pos] = (y, time); orig[pos] = i; hsr[pos] = sector-row
//   k_bin_sort      : orders each bin by original index so the sorted layout is run-to-run deterministic
//                     (atomic ranks are not); results never depend on it -- every tie-break is on `orig`.
#pragma once
#include "common.cuh"

namespace tpc {

// A cluster is inside the geometry iff row is an integer in [0, n_sr), pad in [-0.5, n_pads-0.5) and
// time in [0, max_time]; evaluated in fp32 on the raw values (DESIGN.md §3 C1).
__device__ __forceinline__ bool cluster_key(float rf, float pad, float time, const Consts& c, int& sr, int& bin) {
  bool ok = rf >= 0.0f && rf < (float)c.n_sr && rf == floorf(rf);
  if (!ok) return false;
  sr = (int)rf;
  const int r = sr % c.n_rows;
  ok = pad >= -0.5f && pad < (float)__ldg(c.npads + r) - 0.5f && time >= 0.0f && time <= c.max_time;
  if (!ok) return false;
  bin = sr * c.n_tb + time_bin(time, c);
  return true;
}

__global__ void __launch_bounds__(256) k_ingest_count(const float* __restrict__ row, const float* __restrict__ pad,
                                                      const float* __restrict__ time, int64_t n,
                                                      uint32_t* __restrict__ bin_count, uint32_t* __restrict__ rank,
                                                      uint32_t* __restrict__ n_invalid, const __grid_constant__ Consts c) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  uint32_t bad = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    int sr, bin;
    if (cluster_key(row[i], pad[i], time[i], c, sr, bin)) {
      rank[i] = atomicAdd(bin_count + bin, 1u);
    } else {
      rank[i] = kInvalidRank;
      ++bad;
    }
  }
  bad = __reduce_add_sync(0xffffffffu, bad);
  if (bad && lane_id() == 0) atomicAdd(n_invalid, bad);
}

__global__ void __launch_bounds__(256) k_ingest_scatter(const float* __restrict__ row, const float* __restrict__ pad,
                                                        const float* __restrict__ time, int64_t n,
                                                        const uint32_t* __restrict__ rank, const uint32_t* __restrict__ bin_start,
                                                        float2* __restrict__ yt, uint32_t* __restrict__ orig,
                                                        uint16_t* __restrict__ hsr, const __grid_constant__ Consts c) {
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
    const uint32_t rk = rank[i];
    if (rk == kInvalidRank) continue;
    const float p = pad[i], t = time[i];
    int sr, bin;
    cluster_key(row[i], p, t, c, sr, bin);
    const uint32_t pos = __ldg(bin_start + bin) + rk;
    const float y = (p - __ldg(c.cr + sr % c.n_rows)) * c.P;     // y(h) = (pad - c_r) * P
    yt[pos] = make_float2(y, t);
    orig[pos] = (uint32_t)i;
    hsr[pos] = (uint16_t)sr;
  }
}

// One thread per grid bin: insertion sort of the bin's entries by original index (bins hold a few hits).
__global__ void __launch_bounds__(256) k_bin_sort(const uint32_t* __restrict__ bin_start, float2* __restrict__ yt,
                                                  uint32_t* __restrict__ orig, int n_bins) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= n_bins) return;
  const uint32_t lo = bin_start[b], hi = bin_start[b + 1];
  for (uint32_t i = lo + 1; i < hi; ++i) {
    const uint32_t o = orig[i];
    const float2 v = yt[i];
    uint32_t j = i;
    while (j > lo && orig[j - 1] > o) { orig[j] = orig[j - 1]; yt[j] = yt[j - 1]; --j; }
    if (j != i) { orig[j] = o; yt[j] = v; }
  }
}

}  // namespace tpc
