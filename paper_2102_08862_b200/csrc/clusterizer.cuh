// C0 TPC cluster finder (the step in front of the tracking path; clusterization is
// part of the synchronous GPU load; zero suppression happens in the readout).  Definition: DESIGN.md §3 "C0",
// readings D1..D6 -- a sample is a PEAK iff its ADC reaches the threshold and it beats its (up to) 8 neighbours in
// (pad, time) of the same sector-row (larger ADC, ties to the earlier sample); the cluster of a peak is the centre of
// gravity of its 3 x 3 window, summed in fp32 in the stated order.
//
// Input: samples sorted by (sector_row, time bin, pad).  A GROUP = the samples of one (sector_row, time bin), contiguous
// and pad-sorted, so
//   * the neighbours in the same time bin are the samples at i - 1 / i + 1 (if their pad differs by one),
//   * the time bin before / after is the group before / after (if it has the same sector_row and time +- 1), where the
//     pads p-1, p, p+1 are at most three consecutive entries found by a short binary search.
// Steps: group heads -> exclusive scan = group number of every sample -> group start table -> peak flags -> scan ->
// clusters written in input order (deterministic compaction, no atomics).  One sample per thread; the neighbour reads hit
// L1 / L2 (a sample is read by up to 9 threads of nearby warps).  Algorithmic HBM bytes: 16 per sample read + 16 per
// cluster written (+ scratch: head flag, group number, peak flag / position per sample; three parked sums per peak).
// All arithmetic fp32 in the written order (--fmad=false).
#pragma once
#include "common.cuh"
#include "scan.cuh"

namespace tpc {

struct CfDigits { const int32_t* row; const int32_t* pad; const int32_t* time; const float* adc; };

__global__ void __launch_bounds__(256) k_cf_heads(CfDigits d, int64_t n, uint32_t* __restrict__ head) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  head[i] = (i == 0 || d.row[i] != d.row[i - 1] || d.time[i] != d.time[i - 1]) ? 1u : 0u;
}

// gnum = exclusive scan of head: sample i belongs to group gnum[i] + head[i] - 1; group_start[g] = first sample of group g,
// group_start[n_groups] = n.
__global__ void __launch_bounds__(256) k_cf_groups(const uint32_t* __restrict__ head, const uint32_t* __restrict__ gnum, int64_t n,
                                                   const uint32_t* __restrict__ n_groups, uint32_t* __restrict__ group_start) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) group_start[*n_groups] = (uint32_t)n;
  if (i >= n) return;
  if (head[i]) group_start[gnum[i]] = (uint32_t)i;
}

// The samples of the time bin t + dt of sample i's sector-row that can be in its window: [a, b) holds every sample with
// pad in [p - 1, p + 1] (and at most a few others).  dt = 0: i's own group; dt = +-1: the adjacent group if it is the adjacent
// time bin (a short binary search for the first pad >= p - 1; groups are pad-sorted).
__device__ __forceinline__ void cf_span(const CfDigits& d, const uint32_t* __restrict__ group_start, uint32_t n_groups, int64_t i, uint32_t g,
                                        int dt, int r, int p, int t, int64_t& a, int64_t& b) {
  a = b = 0;
  if (dt == 0) {
    a = max((int64_t)group_start[g], i - 1); b = min((int64_t)group_start[g + 1], i + 2);
    return;
  }
  const int64_t gg = (int64_t)g + dt;
  if (gg < 0 || gg >= (int64_t)n_groups) return;
  const int64_t lo = group_start[gg], hi = group_start[gg + 1];
  if (d.row[lo] != r || d.time[lo] != t + dt) return;           // the adjacent group is not the adjacent time bin
  a = lo; b = hi;
  while (b - a > 3) { const int64_t m = (a + b) >> 1; if (d.pad[m] < p - 1) a = m + 1; else b = m; }
  b = min(hi, a + 6);                                  // the lower bound is within [a, a + 3]; the (up to) three pads follow it
}

struct CfSums { float q, sp, st; };

// One sample per thread: is it a peak (D3, D4)?  A sample at or above the threshold walks its window once, in the order of D5
// (dt outer, dp inner), taking the decision and the three sums together; a peak parks the sums at its own index, so the emit
// kernel needs no neighbour any more.  (Deciding first with early exits -- own time bin, then the adjacent groups -- and
// summing afterwards was measured 3 x slower: the divergent exits cost more than the loads they save.)
__global__ void __launch_bounds__(256) k_cf_peaks(CfDigits d, int64_t n, const uint32_t* __restrict__ head, const uint32_t* __restrict__ gnum,
                                                  const uint32_t* __restrict__ group_start, const uint32_t* __restrict__ n_groups_p,
                                                  float thr, uint32_t* __restrict__ is_peak, CfSums* __restrict__ sums) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const float a0 = d.adc[i];
  bool peak = a0 >= thr;
  if (peak) {
    const uint32_t n_groups = *n_groups_p, g = gnum[i] + head[i] - 1u;
    const int r = d.row[i], p = d.pad[i], t = d.time[i];
    // the window in the order of D5 (dt outer, dp inner): the sums and, on the way, the peak decision
    float q = 0.0f, sp = 0.0f, st = 0.0f;
#pragma unroll
    for (int dt = -1; dt <= 1; ++dt) {
      int64_t a, b;
      cf_span(d, group_start, n_groups, i, g, dt, r, p, t, a, b);
      for (int64_t e = a; e < b; ++e) {
        const int dp = d.pad[e] - p;
        if (dp < -1) continue;
        if (dp > 1) break;
        const float x = d.adc[e];
        if (e != i && !(a0 > x || (a0 == x && i < e))) peak = false;
        q = q + x;
        sp = sp + (float)dp * x;
        st = st + (float)dt * x;
      }
    }
    if (peak) {
      sums[i] = CfSums{q, sp, st};
    }
  }
  is_peak[i] = peak ? 1u : 0u;
}

struct CfOut { int64_t max_clusters; float *row, *pad, *time, *charge; int64_t* n_clusters; int32_t* status; };

// pos = exclusive scan of is_peak (in place); *total behind the last tile offset.  Clusters in the input order of their peaks.
__global__ void __launch_bounds__(256) k_cf_emit(CfDigits d, int64_t n, const uint32_t* __restrict__ pos, const uint32_t* __restrict__ total,
                                                 const CfSums* __restrict__ sums, CfOut o) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    *o.n_clusters = (int64_t)*total;
    *o.status = (int64_t)*total > o.max_clusters ? 1 : 0;       // more clusters than capacity: the first max_clusters are written
  }
  if (i >= n) return;
  const uint32_t k = pos[i];
  const bool mine = (i + 1 < n ? pos[i + 1] : *total) != k;
  if (!mine || (int64_t)k >= o.max_clusters) return;
  const CfSums s = sums[i];
  o.row[k] = (float)d.row[i];
  o.pad[k] = (float)d.pad[i] + s.sp / s.q;
  o.time[k] = (float)d.time[i] + s.st / s.q;
  o.charge[k] = s.q;
}

}  // namespace tpc
