// C2 neighbours finder (BASELINE.json L5 item 2: "one hit per thread with grid lookups in rows r+-1";
// seeding in the time coordinate).  For hit h in row r it forms the candidate sets U (row r+1)
// and D (row r-1) inside the search area |dy| < Ay, |dz| < Az and keeps the pair (u, d) whose second
// differences ey, ez lie inside the window W1 with the smallest mid-point deviation chi2 < chi2_cut
// (DESIGN.md §3 C2).  Ties go to the smallest original index of u, then of d.
//
// Layout: hits sorted by (sector-row, time bin, pad bin); the candidates of one neighbour row are one contiguous span of
// the float2 (y, time) array per grid time bin the search area touches.
// All decision arithmetic is fp32 in the written order, compiled with --fmad=false.
#pragma once
#include "common.cuh"

namespace tpc {

// Pair evaluation shared by the fast path and the overflow fallback: exactly the statement list of C2.
__device__ __forceinline__ void finder_try_pair(const float2 me, const float2 cu, const float2 cd, uint32_t qu, uint32_t qd,
                                                const uint32_t* __restrict__ orig, const Consts& c, float& best, int& bu, int& bd) {
  const float ay = cu.x - me.x;
  const float az = (cu.y - me.y) * c.Z;
  const float by = me.x - cd.x;
  const float ey = ay - by;
  const float bz = (me.y - cd.y) * c.Z;
  const float ez = az - bz;
  if (!(fabsf(ey) < c.W1 && fabsf(ez) < c.W1)) return;
  const float chi2 = (ey * ey) * c.wy + (ez * ez) * c.wz;
  if (!(chi2 < c.chi2_cut)) return;
  bool better = bu < 0 || chi2 < best;
  if (!better && chi2 == best) {                                 // rare: lowest original index wins
    const uint32_t ou = orig[qu], obu = orig[bu];
    better = ou < obu || (ou == obu && orig[qd] < orig[bd]);
  }
  if (better) { best = chi2; bu = (int)qu; bd = (int)qd; }
}

__device__ __forceinline__ bool in_search_area(const float2 me, const float2 cq, const Consts& c) {
  const float dy = cq.x - me.x;
  const float dz = (cq.y - me.y) * c.Z;
  return fabsf(dy) < c.Ay && fabsf(dz) < c.Az;
}

constexpr int kFinderThreads = 256;
#ifndef TPC_FINDER_SLOTS
#define TPC_FINDER_SLOTS 6
#endif
constexpr int kFinderSlots = TPC_FINDER_SLOTS;       // candidates kept per neighbour row in shared memory; more -> generic path

// Scans the candidates of one neighbour row (sector-row srn) inside the search area of hit `me`: for every grid time
// bin the lookup touches, the pad bins pb0..pb1 are one contiguous span (time-major grid, common.cuh::grid_bin).
// Candidates inside the area are appended to the thread's slot list; returns how many were inside (may exceed the slots).
__device__ __forceinline__ int finder_collect(const float2* __restrict__ yt, const uint32_t* __restrict__ bin_start, const float2 me,
                                              int srn, int tb_lo, int tb_hi, int pb0, int pb1, float2 (*s_val)[kFinderThreads],
                                              uint32_t (*s_idx)[kFinderThreads], int slot0, const Consts& c) {
  int n_in = 0;
  for (int tb = tb_lo; tb <= tb_hi; ++tb) {
    const uint32_t b = grid_bin(srn, tb, pb0, c);
    const uint32_t lo = __ldg(bin_start + b), hi = __ldg(bin_start + b + (uint32_t)(pb1 - pb0) + 1u);
    for (uint32_t q = lo; q < hi; ++q) {
      const float2 cq = yt[q];
      if (!in_search_area(me, cq, c)) continue;
      if (n_in < kFinderSlots) { s_val[slot0 + n_in][threadIdx.x] = cq; s_idx[slot0 + n_in][threadIdx.x] = q; }
      ++n_in;
    }
  }
  return n_in;
}

// SIMT shape: the candidates of both neighbour rows that lie inside the search area go to two small per-thread lists in
// shared memory ([slot][thread]: conflict-free); then ONE flat loop over the nu x nd pairs, branch-free apart from the rare
// exact-tie case.  A crowded area (more than kFinderSlots candidates in a row) takes generic nested loops.
__global__ void __launch_bounds__(kFinderThreads) k_neighbours_finder(const float2* __restrict__ yt, const uint32_t* __restrict__ orig,
                                                                      const uint16_t* __restrict__ hsr, const uint32_t* __restrict__ bin_start,
                                                                      int* __restrict__ link_up, int* __restrict__ link_down,
                                                                      const __grid_constant__ Consts c) {
  __shared__ float2 s_val[2 * kFinderSlots][kFinderThreads];      // slots [0, kFinderSlots): up candidates, then down candidates
  __shared__ uint32_t s_idx[2 * kFinderSlots][kFinderThreads];
  const uint32_t n_valid = __ldg(bin_start + c.n_bins);
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_valid) return;
  const int sr = hsr[h];
  const int r = sr % c.n_rows;
  int bu = -1, bd = -1;
  if (r >= 1 && r <= c.n_rows - 2) {
    const float2 me = yt[h];
    const int tb_lo = time_bin(me.y - c.finder_tw, c), tb_hi = time_bin(me.y + c.finder_tw, c);
    const float yo_u = __ldg(c.yoff + r + 1), ps_u = __ldg(c.pscale + r + 1);
    const float yo_d = __ldg(c.yoff + r - 1), ps_d = __ldg(c.pscale + r - 1);
    const int pu0 = pad_bin(me.x - c.finder_yw, yo_u, ps_u, c), pu1 = pad_bin(me.x + c.finder_yw, yo_u, ps_u, c);
    const int pd0 = pad_bin(me.x - c.finder_yw, yo_d, ps_d, c), pd1 = pad_bin(me.x + c.finder_yw, yo_d, ps_d, c);
    const int nu = finder_collect(yt, bin_start, me, sr + 1, tb_lo, tb_hi, pu0, pu1, s_val, s_idx, 0, c);
    const int nd = finder_collect(yt, bin_start, me, sr - 1, tb_lo, tb_hi, pd0, pd1, s_val, s_idx, kFinderSlots, c);
    float best = 0.0f;
    if (nu <= kFinderSlots && nd <= kFinderSlots) {
      const int n_pairs = nu * nd;
      int a = 0, b = 0;
      for (int p = 0; p < n_pairs; ++p) {            // pair (a, b), a-major like the definition's loops
        finder_try_pair(me, s_val[a][threadIdx.x], s_val[kFinderSlots + b][threadIdx.x], s_idx[a][threadIdx.x],
                        s_idx[kFinderSlots + b][threadIdx.x], orig, c, best, bu, bd);
        if (++b == nd) { b = 0; ++a; }
      }
    } else {   // crowded area: generic nested loops over the spans (ties are decided on the original index)
      for (int tu = tb_lo; tu <= tb_hi; ++tu) {
        const uint32_t b_u = grid_bin(sr + 1, tu, pu0, c);
        const uint32_t ulo = __ldg(bin_start + b_u), uhi = __ldg(bin_start + b_u + (uint32_t)(pu1 - pu0) + 1u);
        for (uint32_t qu = ulo; qu < uhi; ++qu) {
          const float2 cu = yt[qu];
          if (!in_search_area(me, cu, c)) continue;
          for (int td = tb_lo; td <= tb_hi; ++td) {
            const uint32_t b_d = grid_bin(sr - 1, td, pd0, c);
            const uint32_t dlo = __ldg(bin_start + b_d), dhi = __ldg(bin_start + b_d + (uint32_t)(pd1 - pd0) + 1u);
            for (uint32_t qd = dlo; qd < dhi; ++qd) {
              const float2 cd = yt[qd];
              if (!in_search_area(me, cd, c)) continue;
              finder_try_pair(me, cu, cd, qu, qd, orig, c, best, bu, bd);
            }
          }
        }
      }
    }
  }
  link_up[h] = bu;
  link_down[h] = bd;
}

}  // namespace tpc
