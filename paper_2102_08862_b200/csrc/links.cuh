// C3 neighbours cleaner + C4 start-hit finder (BASELINE.json L5 item 3: "keeps only reciprocal links ... both
// compacted by warp ballot and scan").  One thread per sorted hit:
//   up'[h]   = u if (u >= 0 and down[u] == h) else -1        (evaluated on the UNCLEANED arrays, written to a
//   down'[h] = d if (d >= 0 and up[d]   == h) else -1         second array -> no race, racecheck-clean)
//   start hit: down'[h] < 0 and the chain h -> up' -> up' ... holds >= seed_min_hits hits.
// Compaction is deterministic: per-CTA counts (ballot popcounts) -> exclusive scan -> ordered write, so the
// start-hit list is in sorted-hit order (sector, row, time bin, original index).
#pragma once
#include "common.cuh"

namespace tpc {

constexpr int kLinkThreads = 256;

__global__ void __launch_bounds__(kLinkThreads) k_clean_links_find_starts(
    const int* __restrict__ link_up, const int* __restrict__ link_down, const uint32_t* __restrict__ bin_start,
    int* __restrict__ link_up_clean, uint8_t* __restrict__ start_flag, uint32_t* __restrict__ cta_count,
    const uint32_t* __restrict__ orig, int32_t* __restrict__ tap_up, int32_t* __restrict__ tap_down,
    uint8_t* __restrict__ tap_start, const __grid_constant__ Consts c) {
  const uint32_t n_valid = __ldg(bin_start + c.n_bins);
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  bool is_start = false;
  if (h < n_valid) {
    const int u = link_up[h], d = link_down[h];
    const int uc = (u >= 0 && link_down[u] == (int)h) ? u : -1;
    const int dc = (d >= 0 && link_up[d] == (int)h) ? d : -1;
    link_up_clean[h] = uc;
    if (dc < 0) {
      int len = 1, cur = (int)h, nxt = uc;
      while (len < c.seed_min_hits && nxt >= 0) {
        cur = nxt; ++len;
        const int uu = link_up[cur];
        nxt = (uu >= 0 && link_down[uu] == cur) ? uu : -1;
      }
      is_start = len >= c.seed_min_hits;
    }
    start_flag[h] = is_start ? 1 : 0;
    if (tap_up) {                                     // parity taps, by original index
      const uint32_t o = orig[h];
      tap_up[o] = uc >= 0 ? (int32_t)orig[uc] : -1;
      tap_down[o] = dc >= 0 ? (int32_t)orig[dc] : -1;
      tap_start[o] = is_start ? 1 : 0;
    }
  }
  const int cnt = __syncthreads_count(is_start);
  if (threadIdx.x == 0) cta_count[blockIdx.x] = (uint32_t)cnt;
}

// cta_offset = exclusive scan of cta_count (cta_offset[n_ctas] = number of start hits).
__global__ void __launch_bounds__(kLinkThreads) k_compact_start_hits(
    const uint8_t* __restrict__ start_flag, const uint32_t* __restrict__ cta_offset, const uint32_t* __restrict__ bin_start,
    uint32_t* __restrict__ start_hits, uint32_t max_tracklets, int n_ctas, int32_t* __restrict__ counters,
    const __grid_constant__ Consts c) {
  __shared__ uint32_t warp_base[kLinkThreads / 32];
  const uint32_t n_valid = __ldg(bin_start + c.n_bins);
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  const bool f = h < n_valid && start_flag[h] != 0;
  const unsigned ballot = __ballot_sync(0xffffffffu, f);
  const int w = threadIdx.x >> 5;
  if (lane_id() == 0) warp_base[w] = __popc(ballot);
  __syncthreads();
  uint32_t base = cta_offset[blockIdx.x];
  for (int i = 0; i < w; ++i) base += warp_base[i];
  if (f) {
    const uint32_t slot = base + __popc(ballot & ((1u << lane_id()) - 1u));
    if (slot < max_tracklets) start_hits[slot] = h;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    const uint32_t total = cta_offset[n_ctas];
    counters[0] = (int32_t)min(total, max_tracklets);     // tracklets actually constructed
    counters[1] = (int32_t)total;                         // start hits found
  }
}

}  // namespace tpc
