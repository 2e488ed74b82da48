// C12 ("Full 5x5 covariance with multiple scattering / energy loss"; §2: the planned
// "improvement of the tracking efficiency, which will require the fit of more tracks and more attached hits").  One inward
// Kalman pass over the hits of every ROOT of the chains linked by C7 (single tracks too): state (y, z, s, t, k) at x, the full
// symmetric 5x5 covariance, process noise from multiple scattering and the mean energy loss of the drift gas.  Definitions:
// DESIGN.md §3 "C12" (readings FF1..FF7).
//
// The covariance lives in 15 registers, named by (row, column) of the lower triangle in the state order (y, z, s, t, k):
//   P00 | P10 P11 | P20 P21 P22 | P30 P31 P32 P33 | P40 P41 P42 P43 P44        (stored in that order: cov15)
// All arithmetic is fp32 in the written order (the translation unit is compiled with --fmad=false); sqrtf and the divisions
// are the IEEE ones.
//
// SIMT mapping as C8's k_refit_chains: persistent warps, one lane per root at a time, lanes refilled from a global counter;
// one loop iteration = one hit (step + two scalar updates), the next hit's coordinates are read one iteration ahead.
#pragma once
#include "merge.cuh"

namespace tpc {

struct FullFitConsts { float inv_x0, dedx_mip, m2, ms2, eloss_sigma; };

struct FullState {
  float x, y, z, s, t, k;
  float P00, P10, P11, P20, P21, P22, P30, P31, P32, P33, P40, P41, P42, P43, P44;
};

struct FullFitIo {
  const float2* hit_yt; const uint8_t* hit_row;
  const int32_t* n_hits; const int64_t* hit_offset; int64_t max_track_hits;
  const int32_t *next, *prev;
  const int32_t *ce_next, *ce_prev; const float* t_ce;   // C10's links (reading FF8); all three nullptr = plain C12
  int32_t *ok, *chain_hits, *chain_pieces;   // [max_tracks]
  float *par7, *cov15;                       // [max_tracks * 7], [max_tracks * 15]
};

// FF8: the piece behind the central electrode that continues piece e, or -1: C10's link counts only where no sector-boundary
// link competes at either end.
__device__ __forceinline__ int fullfit_crosses_into(const FullFitIo& io, int e) {
  if (!io.ce_next || io.next[e] >= 0) return -1;
  const int b = io.ce_next[e];
  return (b >= 0 && io.prev[b] < 0) ? b : -1;
}

// Pass-through values for every track + the list of roots (prev < 0), in any order: results are indexed by track.
__global__ void __launch_bounds__(256) k_fullfit_roots(MergeTracks T, FullFitIo io, uint32_t* __restrict__ root_list,
                                                       uint32_t* __restrict__ n_roots, const __grid_constant__ MergeConsts c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  bool is_root = false;
  if (i < merge_n(T, c)) {
    is_root = io.prev[i] < 0;
    if (is_root && io.ce_next) { const int a = io.ce_prev[i]; if (a >= 0 && fullfit_crosses_into(io, a) == i) is_root = false; }   // continuation of a chain from the other side
    io.ok[i] = 0; io.chain_hits[i] = io.n_hits[i]; io.chain_pieces[i] = 1;
    float* rp = io.par7 + 7 * (size_t)i;
    rp[0] = T.x[i]; rp[1] = T.y[i]; rp[2] = T.z[i]; rp[3] = T.s[i]; rp[4] = T.t[i]; rp[5] = T.k[i]; rp[6] = T.time_ref[i];
    float* rc = io.cov15 + 15 * (size_t)i;
#pragma unroll
    for (int k = 0; k < 15; ++k) rc[k] = 0.0f;
  }
  const unsigned m = __ballot_sync(0xffffffffu, is_root);
  if (m) {
    uint32_t base = 0;
    const int leader = __ffs(m) - 1;
    if ((int)lane_id() == leader) base = atomicAdd(n_roots, (uint32_t)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (is_root) root_list[base + __popc(m & ((1u << lane_id()) - 1u))] = (uint32_t)i;
  }
}

// step = transport of state and covariance to x = xn, then the material of the segment.  false (state unchanged) on FAIL.
__device__ __forceinline__ bool full_step(FullState& S, float xn, float cB, float sin_phi_max, const FullFitConsts& m) {
  const float dx = xn - S.x;
  const float kc = cB * S.k;
  const float sn = S.s + kc * dx;
  if (!(fabsf(S.s) < sin_phi_max && fabsf(sn) < sin_phi_max)) return false;
  const float c = sqrtf(1.0f - S.s * S.s);
  const float cn = sqrtf(1.0f - sn * sn);
  const float ss = S.s + sn;
  const float cc = c + cn;
  const float icc = 1.0f / cc;
  const float T = ss * icc;
  const float q = 1.0f + T * T;
  const float rq = sqrtf(q);
  const float u = kc * dx;
  const float a = (u * u) * q;
  const float dS = (dx * rq) * (1.0f + a * (0.041666668f + a * (0.0046875f + a * 0.00069754466f)));
  const float g0 = (1.0f + T * (S.s / c)) * icc;
  const float g1 = (1.0f + T * (sn / cn)) * icc;
  const float fa = dx * (g0 + g1);
  const float e = cB * dx;
  const float fb = (dx * g1) * e;
  const float gm = S.t * (T / rq);
  const float zs = gm * fa;
  const float zk = gm * fb;
  S.y = S.y + dx * T;
  S.z = S.z + S.t * dS;
  S.s = sn;
  S.x = xn;
  // A = F P: rows y (columns 0, 2, 4 are all that P' needs), z, s; rows t and k of A are those of P
  const float A00 = S.P00 + fa * S.P20 + fb * S.P40;
  const float A02 = S.P20 + fa * S.P22 + fb * S.P42;
  const float A04 = S.P40 + fa * S.P42 + fb * S.P44;
  const float A10 = S.P10 + zs * S.P20 + S.P30 * dS + zk * S.P40;
  const float A11 = S.P11 + zs * S.P21 + S.P31 * dS + zk * S.P41;
  const float A12 = S.P21 + zs * S.P22 + S.P32 * dS + zk * S.P42;
  const float A13 = S.P31 + zs * S.P32 + S.P33 * dS + zk * S.P43;
  const float A14 = S.P41 + zs * S.P42 + S.P43 * dS + zk * S.P44;
  const float A20 = S.P20 + e * S.P40;
  const float A21 = S.P21 + e * S.P41;
  const float A22 = S.P22 + e * S.P42;
  const float A23 = S.P32 + e * S.P43;
  const float A24 = S.P42 + e * S.P44;
  // P' = A F^T, lower triangle
  S.P00 = A00 + fa * A02 + fb * A04;
  S.P10 = A10 + fa * A12 + fb * A14;
  S.P11 = A11 + zs * A12 + A13 * dS + zk * A14;
  S.P20 = A20 + fa * A22 + fb * A24;
  S.P21 = A21 + zs * A22 + A23 * dS + zk * A24;
  S.P22 = A22 + e * A24;
  const float n30 = S.P30 + fa * S.P32 + fb * S.P43;
  const float n31 = S.P31 + zs * S.P32 + S.P33 * dS + zk * S.P43;
  const float n32 = S.P32 + e * S.P43;
  const float n40 = S.P40 + fa * S.P42 + fb * S.P44;
  const float n41 = S.P41 + zs * S.P42 + S.P43 * dS + zk * S.P44;
  const float n42 = S.P42 + e * S.P44;
  S.P30 = n30; S.P31 = n31; S.P32 = n32;
  S.P40 = n40; S.P41 = n41; S.P42 = n42;
  // material of the segment (t and k are the values the transport used, s the new one)
  const float tt1 = 1.0f + S.t * S.t;
  const float Lp = fabsf(dS) * sqrtf(tt1);
  const float ip2 = (S.k * S.k) / tt1;
  const float ib2 = 1.0f + m.m2 * ip2;
  const float ibp2 = ip2 * ib2;
  const float th2 = (m.ms2 * ibp2) * (Lp * m.inv_x0);
  S.P22 = S.P22 + th2 * ((1.0f - sn * sn) * tt1);
  S.P33 = S.P33 + th2 * (tt1 * tt1);
  const float tk = S.t * S.k;
  S.P43 = S.P43 + th2 * (tk * tt1);
  S.P44 = S.P44 + th2 * (tk * tk);
  const float dl = ((m.dedx_mip * ib2) * Lp) * sqrtf(ibp2);
  S.k = S.k * (1.0f - dl);
  const float ek = (S.k * dl) * m.eloss_sigma;
  S.P44 = S.P44 + ek * ek;
  return true;
}

// Scalar measurement of y (variance ry), then of z (variance rz); each: gain = column / (variance + r), state and the lower
// triangle are updated with the OLD column.
__device__ __forceinline__ void full_update(FullState& S, float ym, float zm, float ry, float rz) {
  {
    const float c0 = S.P00, c1 = S.P10, c2 = S.P20, c3 = S.P30, c4 = S.P40;
    const float w = 1.0f / (c0 + ry);
    const float res = ym - S.y;
    const float K0 = c0 * w, K1 = c1 * w, K2 = c2 * w, K3 = c3 * w, K4 = c4 * w;
    S.y = S.y + K0 * res; S.z = S.z + K1 * res; S.s = S.s + K2 * res; S.t = S.t + K3 * res; S.k = S.k + K4 * res;
    S.P00 = S.P00 - K0 * c0;
    S.P10 = S.P10 - K1 * c0; S.P11 = S.P11 - K1 * c1;
    S.P20 = S.P20 - K2 * c0; S.P21 = S.P21 - K2 * c1; S.P22 = S.P22 - K2 * c2;
    S.P30 = S.P30 - K3 * c0; S.P31 = S.P31 - K3 * c1; S.P32 = S.P32 - K3 * c2; S.P33 = S.P33 - K3 * c3;
    S.P40 = S.P40 - K4 * c0; S.P41 = S.P41 - K4 * c1; S.P42 = S.P42 - K4 * c2; S.P43 = S.P43 - K4 * c3; S.P44 = S.P44 - K4 * c4;
  }
  {
    const float c0 = S.P10, c1 = S.P11, c2 = S.P21, c3 = S.P31, c4 = S.P41;
    const float w = 1.0f / (c1 + rz);
    const float res = zm - S.z;
    const float K0 = c0 * w, K1 = c1 * w, K2 = c2 * w, K3 = c3 * w, K4 = c4 * w;
    S.y = S.y + K0 * res; S.z = S.z + K1 * res; S.s = S.s + K2 * res; S.t = S.t + K3 * res; S.k = S.k + K4 * res;
    S.P00 = S.P00 - K0 * c0;
    S.P10 = S.P10 - K1 * c0; S.P11 = S.P11 - K1 * c1;
    S.P20 = S.P20 - K2 * c0; S.P21 = S.P21 - K2 * c1; S.P22 = S.P22 - K2 * c2;
    S.P30 = S.P30 - K3 * c0; S.P31 = S.P31 - K3 * c1; S.P32 = S.P32 - K3 * c2; S.P33 = S.P33 - K3 * c3;
    S.P40 = S.P40 - K4 * c0; S.P41 = S.P41 - K4 * c1; S.P42 = S.P42 - K4 * c2; S.P43 = S.P43 - K4 * c3; S.P44 = S.P44 - K4 * c4;
  }
}

__device__ __forceinline__ void full_reset(FullState& S, const Consts& tc) {
  S.P00 = tc.c0_y2; S.P11 = tc.c0_z2; S.P22 = tc.c0_s2; S.P33 = tc.c0_t2; S.P44 = tc.c0_k2;
  S.P10 = S.P20 = S.P21 = S.P30 = S.P31 = S.P32 = S.P40 = S.P41 = S.P42 = S.P43 = 0.0f;
}

constexpr int kFullFitRefill = 4;
__global__ void __launch_bounds__(kMergeThreads) k_refit_full(MergeTracks T, FullFitIo io, const uint32_t* __restrict__ root_list,
                                                               const uint32_t* __restrict__ n_roots, uint32_t* __restrict__ work_counter,
                                                               const __grid_constant__ MergeConsts c, const __grid_constant__ Consts tc,
                                                               const __grid_constant__ FullFitConsts m) {
  __shared__ float xr[kRowStride];
  for (int r = threadIdx.x; r < tc.n_rows; r += blockDim.x) xr[r] = tc.xr[r];
  __syncthreads();
  const uint32_t n_work = *n_roots;
  const unsigned lane = lane_id();
  bool active = false, exhausted = false;
  int root = -1, p = -1;
  int64_t j = 0, off = 0;
  float tref = 0.0f;
  float2 hy = make_float2(0.0f, 0.0f);                 // (y, time) of the current hit
  int hr = 0;                                          // its pad row
  FullState S;
  S.x = S.y = S.z = S.s = S.t = S.k = 0.0f;
  full_reset(S, tc);
  for (;;) {
    const unsigned idle = __ballot_sync(0xffffffffu, !active && !exhausted);
    const unsigned busy = __ballot_sync(0xffffffffu, active);
    if (idle && (__popc(idle) >= kFullFitRefill || busy == 0)) {
      if (!active && !exhausted) {
        const uint32_t e = (uint32_t)take_tracklets(work_counter, idle, lane);
        if (e >= n_work) {
          exhausted = true;
        } else {
          root = (int)root_list[e];
          int pm = root, pieces = 1, total = io.n_hits[root];
          bool complete = io.n_hits[root] > 0 && io.hit_offset[root] + io.n_hits[root] <= io.max_track_hits;   // list not cut by TPC_STATUS_TRACK_HIT_OVERFLOW
          bool crossed = false;
          for (;;) {
            int q = io.next[pm];
            if (q < 0 && !crossed) { q = fullfit_crosses_into(io, pm); crossed = q >= 0; }       // FF8: once, behind the electrode
            if (q < 0) break;
            if (pieces >= 4 * c.n_rows) { complete = false; break; }      // cannot happen (M7); never walk a corrupted link list for ever
            pm = q; ++pieces; total += io.n_hits[q];
            complete = complete && io.n_hits[q] > 0 && io.hit_offset[q] + io.n_hits[q] <= io.max_track_hits;
          }
          io.chain_hits[root] = total;
          io.chain_pieces[root] = pieces;
          p = pm; off = io.hit_offset[pm]; j = off + io.n_hits[pm] - 1; tref = T.time_ref[pm];
          if (complete) { hy = io.hit_yt[j]; hr = io.hit_row[j]; } else { hr = 0; }
          // FF1: the outermost piece's state goes to its outermost hit with the plain C5 transport, then the reset covariance
          TrackState S0;
          S0.x = T.x[pm]; S0.y = T.y[pm]; S0.z = T.z[pm]; S0.s = T.s[pm]; S0.t = T.t[pm]; S0.k = T.k[pm];
          S0.c0 = S0.c1 = S0.c2 = S0.c3 = S0.c4 = S0.c5 = 0.0f; S0.d0 = S0.d1 = S0.d2 = 0.0f;
          const bool ok0 = transport(S0, xr[hr], tc.cB, tc.sin_phi_max);
          S.x = S0.x; S.y = S0.y; S.z = S0.z; S.s = S0.s; S.t = S0.t; S.k = S0.k;
          full_reset(S, tc);
          if (ok0 && complete) active = true; else io.ok[root] = -1;
        }
      }
    }
    if (busy == 0 && __ballot_sync(0xffffffffu, active) == 0) {
      if (__ballot_sync(0xffffffffu, !exhausted) == 0) break;
      continue;
    }
    if (active) {
      float2 ny = make_float2(0.0f, 0.0f);
      int nr = 0;
      if (j > off) { ny = io.hit_yt[j - 1]; nr = io.hit_row[j - 1]; }      // the next hit, one iteration ahead
      bool good = full_step(S, xr[hr], tc.cB, tc.sin_phi_max, m);
      if (good) {
        full_update(S, hy.x, (hy.y - tref) * tc.Z, tc.ry, tc.rz);
        if (j > off) {
          --j; hy = ny; hr = nr;
        } else if (p == root) {                        // innermost hit of the root piece: done
          io.ok[root] = 1;
          float* rp = io.par7 + 7 * (size_t)root;
          rp[0] = S.x; rp[1] = S.y; rp[2] = S.z; rp[3] = S.s; rp[4] = S.t; rp[5] = S.k;      // rp[6] = time_ref of the root: already there
          float* rc = io.cov15 + 15 * (size_t)root;
          rc[0] = S.P00; rc[1] = S.P10; rc[2] = S.P11; rc[3] = S.P20; rc[4] = S.P21; rc[5] = S.P22; rc[6] = S.P30; rc[7] = S.P31;
          rc[8] = S.P32; rc[9] = S.P33; rc[10] = S.P40; rc[11] = S.P41; rc[12] = S.P42; rc[13] = S.P43; rc[14] = S.P44;
          active = false;
        } else if (io.prev[p] < 0) {                   // the central electrode (FF8): reflect the time coordinate about t_ce, no rotation
          const int pin = io.ce_prev[p];
          const float tce = io.t_ce[pin], tref_in = T.time_ref[pin];
          S.z = (((tce + tce) - tref) - tref_in) * tc.Z - S.z;
          S.t = -S.t;
          S.P10 = -S.P10; S.P21 = -S.P21; S.P30 = -S.P30; S.P32 = -S.P32; S.P41 = -S.P41; S.P43 = -S.P43;
          p = pin; tref = tref_in; off = io.hit_offset[pin]; j = off + io.n_hits[pin] - 1;
          hy = io.hit_yt[j]; hr = io.hit_row[j];
        } else {                                       // piece boundary: rotate into the frame of the next inner piece
          const int pin = io.prev[p];
          const float sg = ((T.sector[p] % 18) == ((T.sector[pin] % 18) + 1) % 18) ? 1.0f : -1.0f;
          const float qd = -sg;
          const float cs = sqrtf(1.0f - S.s * S.s);
          const float J = c.Cd + qd * ((S.s / cs) * c.Sd);
          const float x1 = S.x * c.Cd + qd * (S.y * c.Sd);
          const float y1 = S.y * c.Cd - qd * (S.x * c.Sd);
          const float s1 = S.s * c.Cd - qd * (cs * c.Sd);
          if (fabsf(s1) < tc.sin_phi_max) {
            S.x = x1; S.y = y1; S.s = s1;
            S.P20 = S.P20 * J; S.P21 = S.P21 * J; S.P32 = S.P32 * J; S.P42 = S.P42 * J;
            S.P22 = (S.P22 * J) * J;
            const float tref_in = T.time_ref[pin];
            S.z = S.z + (tref - tref_in) * tc.Z;
            p = pin; tref = tref_in; off = io.hit_offset[pin]; j = off + io.n_hits[pin] - 1;
            hy = io.hit_yt[j]; hr = io.hit_row[j];
          } else {
            good = false;
          }
        }
      }
      if (!good) { io.ok[root] = -1; active = false; }
    }
  }
}

}  // namespace tpc
