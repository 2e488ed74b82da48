// C3 neighbours cleaner + C4 start-hit finder (BASELINE.json L5 item 3: "keeps only reciprocal links ... both
// compacted by warp ballot and scan").  One thread per sorted hit:
//   up'[h]   = u if (u >= 0 and down[u] == h) else -1        (evaluated on the UNCLEANED arrays, written to a
//   down'[h] = d if (d >= 0 and up[d]   == h) else -1         second array -> no race, racecheck-clean)
//   start hit: down'[h] < 0 and the chain h -> up' -> up' ... holds >= seed_min_hits hits.
// Compaction is deterministic: per-cell counts -> exclusive scan -> ordered write (see below).
#pragma once
#include "common.cuh"

namespace tpc {

constexpr int kLinkThreads = 256;

__global__ void __launch_bounds__(kLinkThreads) k_clean_links_find_starts(
    const int* __restrict__ link_up, const int* __restrict__ link_down, const uint32_t* __restrict__ bin_start,
    int* __restrict__ link_up_clean, uint8_t* __restrict__ start_flag,
    const uint32_t* __restrict__ orig, int32_t* __restrict__ tap_up, int32_t* __restrict__ tap_down,
    uint8_t* __restrict__ tap_start, const __grid_constant__ Consts c) {
  const uint32_t n_valid = __ldg(bin_start + c.n_bins);
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h < n_valid) {
    bool is_start = false;
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
}

// Start-hit compaction in PROCESSING order.  The constructor's in-flight tracklets should be close in space and
// time so that the hits and grid bins they touch stay in L2: start hits are therefore listed by
// (sector, time slice, row) instead of the hits' own (sector, row, time) order.  A cell (sector, slice, row) is one
// contiguous range of sorted hits (the grid is time-major inside a sector-row), so the compaction is: one thread per cell
// counts its flags -> exclusive scan over the cells in processing order -> the same thread writes its start hits.
// Deterministic (no atomics).
struct StartCells { int n_slices, slice_bins; uint32_t n_cells; };   // slice_bins: grid time bins per slice

__device__ __forceinline__ void start_cell_range(uint32_t cell, const StartCells sc, const uint32_t* __restrict__ bin_start,
                                                 const Consts& c, uint32_t& lo, uint32_t& hi) {
  const int r = (int)(cell % (uint32_t)c.n_rows);
  const uint32_t q = cell / (uint32_t)c.n_rows;
  const int slice = (int)(q % (uint32_t)sc.n_slices);
  const int sector = (int)(q / (uint32_t)sc.n_slices);
  const int sr = sector * c.n_rows + r;
  const int t0 = slice * sc.slice_bins;
  lo = __ldg(bin_start + grid_bin(sr, t0, 0, c));
  hi = __ldg(bin_start + grid_bin(sr, min(t0 + sc.slice_bins, c.n_tb), 0, c));      // (sr, n_tb, 0) == (sr + 1, 0, 0)
}

__global__ void __launch_bounds__(kLinkThreads) k_start_cell_count(const uint8_t* __restrict__ start_flag,
                                                                   const uint32_t* __restrict__ bin_start, StartCells sc,
                                                                   uint32_t* __restrict__ cell_count, const __grid_constant__ Consts c) {
  const uint32_t cell = blockIdx.x * blockDim.x + threadIdx.x;
  if (cell >= sc.n_cells) return;
  uint32_t lo, hi;
  start_cell_range(cell, sc, bin_start, c, lo, hi);
  uint32_t cnt = 0;
  for (uint32_t h = lo; h < hi; ++h) cnt += start_flag[h];
  cell_count[cell] = cnt;
}

// cell_offset = exclusive scan of cell_count; *total = number of start hits.
__global__ void __launch_bounds__(kLinkThreads) k_start_cell_write(const uint8_t* __restrict__ start_flag,
                                                                   const uint32_t* __restrict__ bin_start, StartCells sc,
                                                                   const uint32_t* __restrict__ cell_offset, const uint32_t* __restrict__ total,
                                                                   uint32_t* __restrict__ start_hits, uint32_t max_tracklets,
                                                                   int32_t* __restrict__ counters, const __grid_constant__ Consts c) {
  const uint32_t cell = blockIdx.x * blockDim.x + threadIdx.x;
  if (cell == 0) {
    counters[0] = (int32_t)min(*total, max_tracklets);     // tracklets actually constructed
    counters[1] = (int32_t)*total;                         // start hits found
  }
  if (cell >= sc.n_cells) return;
  uint32_t lo, hi;
  start_cell_range(cell, sc, bin_start, c, lo, hi);
  uint32_t slot = cell_offset[cell];
  for (uint32_t h = lo; h < hi; ++h)
    if (start_flag[h]) { if (slot < max_tracklets) start_hits[slot] = h; ++slot; }
}

}  // namespace tpc
