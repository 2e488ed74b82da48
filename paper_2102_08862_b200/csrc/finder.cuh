// C2 neighbours finder (BASELINE.json L5 item 2: "one hit per thread with grid lookups in rows r+-1";
// seeding in the time coordinate).  For hit h in row r it forms the candidate sets U (row r+1)
// and D (row r-1) inside the search area |dy| < Ay, |dz| < Az and keeps the pair (u, d) whose second
// differences ey, ez lie inside the window W1 with the smallest mid-point deviation chi2 < chi2_cut
// (DESIGN.md §3 C2).  Ties go to the smallest original index of u, then of d.
//
// Layout: hits sorted by (sector-row, time bin); the candidates of one neighbour row are ONE contiguous span
// [binStart[b(t-A)], binStart[b(t+A)+1]) of the float2 (y, time) array, so a thread streams ~64 B per row.
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

// SIMT shape: ONE flat loop scans the candidates of both neighbour rows and keeps those inside the search area
// in register slots (<= 4 per row; more is rare and takes the generic nested loop), then a short pair loop.
// The nested "for u: for d" form ran at 4.5 of 32 lanes (profiles/r01a_ncu_full_baseline.md).
__global__ void __launch_bounds__(256) k_neighbours_finder(const float2* __restrict__ yt, const uint32_t* __restrict__ orig,
                                                           const uint16_t* __restrict__ hsr, const uint32_t* __restrict__ bin_start,
                                                           int* __restrict__ link_up, int* __restrict__ link_down,
                                                           const __grid_constant__ Consts c) {
  const uint32_t n_valid = __ldg(bin_start + c.n_bins);
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_valid) return;
  const int sr = hsr[h];
  const int r = sr % c.n_rows;
  int bu = -1, bd = -1;
  if (r >= 1 && r <= c.n_rows - 2) {
    const float2 me = yt[h];
    const int tb_lo = time_bin(me.y - c.finder_tw, c), tb_hi = time_bin(me.y + c.finder_tw, c);
    const uint32_t* bs_u = bin_start + (size_t)(sr + 1) * c.n_tb;
    const uint32_t* bs_d = bin_start + (size_t)(sr - 1) * c.n_tb;
    const uint32_t u_lo = __ldg(bs_u + tb_lo), u_hi = __ldg(bs_u + tb_hi + 1);
    const uint32_t d_lo = __ldg(bs_d + tb_lo), d_hi = __ldg(bs_d + tb_hi + 1);
    const uint32_t n_u = u_hi - u_lo, n_all = n_u + (d_hi - d_lo);
    uint32_t us0 = 0, us1 = 0, us2 = 0, us3 = 0, ds0 = 0, ds1 = 0, ds2 = 0, ds3 = 0;
    int nu = 0, nd = 0;
    for (uint32_t ib = 0; ib < n_all; ib += 4) {     // batches of 4 independent loads
      float2 cq[4];
      uint32_t qq[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t i = min(ib + k, n_all - 1);
        qq[k] = i < n_u ? u_lo + i : d_lo + (i - n_u);
        cq[k] = yt[qq[k]];
      }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t i = ib + k;
        if (!(i < n_all && in_search_area(me, cq[k], c))) continue;
        const uint32_t q = qq[k];
        if (i < n_u) {
          if (nu == 0) us0 = q; else if (nu == 1) us1 = q; else if (nu == 2) us2 = q; else if (nu == 3) us3 = q;
          ++nu;
        } else {
          if (nd == 0) ds0 = q; else if (nd == 1) ds1 = q; else if (nd == 2) ds2 = q; else if (nd == 3) ds3 = q;
          ++nd;
        }
      }
    }
    float best = 0.0f;
    if (nu <= 4 && nd <= 4) {
      for (int a = 0; a < nu; ++a) {
        const uint32_t qu = a == 0 ? us0 : a == 1 ? us1 : a == 2 ? us2 : us3;
        const float2 cu = yt[qu];
        for (int b = 0; b < nd; ++b) {
          const uint32_t qd = b == 0 ? ds0 : b == 1 ? ds1 : b == 2 ? ds2 : ds3;
          finder_try_pair(me, cu, yt[qd], qu, qd, orig, c, best, bu, bd);
        }
      }
    } else {   // crowded area: generic nested loops over the spans, same pair order
      for (uint32_t qu = u_lo; qu < u_hi; ++qu) {
        const float2 cu = yt[qu];
        if (!in_search_area(me, cu, c)) continue;
        for (uint32_t qd = d_lo; qd < d_hi; ++qd) {
          const float2 cd = yt[qd];
          if (!in_search_area(me, cd, c)) continue;
          finder_try_pair(me, cu, cd, qu, qd, orig, c, best, bu, bd);
        }
      }
    }
  }
  link_up[h] = bu;
  link_down[h] = bd;
}

}  // namespace tpc
