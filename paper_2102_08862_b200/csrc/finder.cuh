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

// Candidate span of one (sector-row, pad bin): the hits of the time bins [tb_lo, tb_hi].
struct Span { uint32_t lo, n; };
__device__ __forceinline__ Span grid_span(const uint32_t* __restrict__ bin_start, int sr, int pb, int tb_lo, int tb_hi, const Consts& c) {
  const uint32_t* bs = bin_start + ((size_t)sr * c.n_pb + pb) * c.n_tb;
  const uint32_t lo = __ldg(bs + tb_lo);
  return Span{lo, __ldg(bs + tb_hi + 1) - lo};
}

constexpr int kFinderThreads = 256;
#ifndef TPC_FINDER_SLOTS
#define TPC_FINDER_SLOTS 6
#endif
constexpr int kFinderSlots = TPC_FINDER_SLOTS;       // candidates kept per neighbour row in shared memory; more -> generic path

// SIMT shape: (1) ONE flat loop scans the candidates of both neighbour rows (each row: the spans of one or two pad
// bins -- the create-time check guarantees that the search area is narrower than a pad bin) and appends those inside
// the search area to two small per-thread lists in shared memory ([slot][thread]: conflict-free); (2) ONE flat loop
// over the nu x nd pairs.  Both trip counts are the maximum over the warp of a small number, and the bodies are
// branch-free apart from the rare exact-tie case.  The nested "for u: for d" form over the raw spans ran at 4.5 of
// 32 lanes (round-1 ncu capture).
__global__ void __launch_bounds__(kFinderThreads) k_neighbours_finder(const float2* __restrict__ yt, const uint32_t* __restrict__ orig,
                                                                      const uint16_t* __restrict__ hsr, const uint32_t* __restrict__ bin_start,
                                                                      int* __restrict__ link_up, int* __restrict__ link_down,
                                                                      const __grid_constant__ Consts c) {
  __shared__ float2 s_val[2 * kFinderSlots][kFinderThreads];      // rows 0..3: up candidates, 4..7: down candidates
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
    // spans: u0, u1 (row r+1), d0, d1 (row r-1); the second span of a row is empty unless the area straddles two pad bins
    const Span u0 = grid_span(bin_start, sr + 1, pu0, tb_lo, tb_hi, c);
    const Span d0 = grid_span(bin_start, sr - 1, pd0, tb_lo, tb_hi, c);
    Span u1{0u, 0u}, d1{0u, 0u};
    if (pu1 != pu0) u1 = grid_span(bin_start, sr + 1, pu1, tb_lo, tb_hi, c);
    if (pd1 != pd0) d1 = grid_span(bin_start, sr - 1, pd1, tb_lo, tb_hi, c);
    const uint32_t e0 = u0.n, e1 = e0 + u1.n, e2 = e1 + d0.n, n_all = e2 + d1.n;   // up candidates: i < e1
    // flat index i -> sorted-hit index: base of the span that holds i, minus the span's first i
    const uint32_t b0 = u0.lo, b1 = u1.lo - e0, b2 = d0.lo - e1, b3 = d1.lo - e2;
    int nu = 0, nd = 0;
    for (uint32_t ib = 0; ib < n_all; ib += 2) {     // two independent loads per trip
      uint32_t qq[2];
      float2 cq[2];
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const uint32_t i = min(ib + k, n_all - 1);
        qq[k] = (i < e1 ? (i < e0 ? b0 : b1) : (i < e2 ? b2 : b3)) + i;
        cq[k] = yt[qq[k]];
      }
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        const uint32_t i = ib + k;
        if (i < n_all && in_search_area(me, cq[k], c)) {
          const bool up = i < e1;
          const int slot = up ? nu : kFinderSlots + nd;
          if ((up ? nu : nd) < kFinderSlots) { s_val[slot][threadIdx.x] = cq[k]; s_idx[slot][threadIdx.x] = qq[k]; }
          nu += up ? 1 : 0;
          nd += up ? 0 : 1;
        }
      }
    }
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
      auto index_of = [&](uint32_t i) -> uint32_t { return (i < e1 ? (i < e0 ? b0 : b1) : (i < e2 ? b2 : b3)) + i; };
      for (uint32_t iu = 0; iu < e1; ++iu) {
        const uint32_t qu = index_of(iu);
        const float2 cu = yt[qu];
        if (!in_search_area(me, cu, c)) continue;
        for (uint32_t id = e1; id < n_all; ++id) {
          const uint32_t qd = index_of(id);
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
