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
    float best = 0.0f;
    for (uint32_t qu = u_lo; qu < u_hi; ++qu) {
      const float2 cu = yt[qu];
      const float ay = cu.x - me.x;
      const float az = (cu.y - me.y) * c.Z;
      if (!(fabsf(ay) < c.Ay && fabsf(az) < c.Az)) continue;          // u in U
      for (uint32_t qd = d_lo; qd < d_hi; ++qd) {
        const float2 cd = yt[qd];
        const float dyd = cd.x - me.x;
        const float dzd = (cd.y - me.y) * c.Z;
        if (!(fabsf(dyd) < c.Ay && fabsf(dzd) < c.Az)) continue;      // d in D
        const float by = me.x - cd.x;
        const float ey = ay - by;
        const float bz = (me.y - cd.y) * c.Z;
        const float ez = az - bz;
        if (!(fabsf(ey) < c.W1 && fabsf(ez) < c.W1)) continue;
        const float chi2 = (ey * ey) * c.wy + (ez * ez) * c.wz;
        if (!(chi2 < c.chi2_cut)) continue;
        bool better = bu < 0 || chi2 < best;
        if (!better && chi2 == best) {                                 // rare: lowest original index wins
          const uint32_t ou = orig[qu], obu = orig[bu];
          better = ou < obu || (ou == obu && orig[qd] < orig[bd]);
        }
        if (better) { best = chi2; bu = (int)qu; bd = (int)qd; }
      }
    }
  }
  link_up[h] = bu;
  link_down[h] = bd;
}

}  // namespace tpc
