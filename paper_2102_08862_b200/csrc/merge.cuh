// C7 sector-boundary merging of the per-sector tracks (DESIGN.md §3 "C7", readings M1..M8; "full TPC
// tracking" -- the per-sector tracker is followed by a merger of the sector tracks; BASELINE.json L8: 36 sectors, each in
// its rotated local frame).
//
// A track A is rotated into the frame of each neighbour sector (same side, +-20 degrees), transported to every pad row
// r_B of the row window, and compared with the tracks B of that sector whose state sits on row r_B: reciprocal best
// match in d2 = dy^2 wy + dz^2 wz + ds^2 ws + dk^2 wk inside the four cuts, every tie -> lowest seed id.
//
// Layout: the tracks are binned by (sector, state row, 32-time-bin cell of the state's time) with a counting sort
// (histogram -> exclusive scan -> fill); the candidate records (y, z_rel, sin phi, q/pT | time_ref, seed) are stored in
// cell order, so the candidates of one (row, time window) are one contiguous span.  One thread per track A: two
// rotations, one state transport per row of the window (it serves every candidate of that row), a few candidates per
// row.  in[B] is a 64-bit atomicMin on (d2 bits, seed of A) -- d2 >= 0, so its bit pattern orders like its value -- and
// out[A] the same key kept in a register: the result does not depend on the order in which candidates are met.
// All decision arithmetic is fp32 in the written order (--fmad=false).
#pragma once
#include "common.cuh"
#include "tracklet.cuh"

namespace tpc {

constexpr int kMergeThreads = 128;
constexpr int kMergeCellTimeBins = 32;

struct MergeConsts {
  int n_sectors, n_rows, n_tcell, gap, overlap, max_tracks;
  float x0, pitch, Cd, Sd, Z, inv_Z, cB, sin_phi_max;
  float cut_y, cut_z, cut_s, cut_k, wy, wz, ws, wk;
  float inv_cell, t_window;      // 1 / kMergeCellTimeBins; half width of the time lookup = cut_z / Z + 0.5 bins
  const float* xr;               // [n_rows] x of the pad row (the handle's table)
};

struct MergeTracks {   // device pointers of tpc_tracks_t
  const int32_t *n_tracks, *seed, *sector, *first_row, *last_row;
  const float *x, *y, *z, *time_ref, *s, *t, *k;
};

struct MergeScratch {
  uint32_t* cell_start;          // [n_cells + 1] histogram, then its exclusive scan
  uint32_t* cell_cursor;         // [n_cells]
  uint32_t* cell_of;             // [max_tracks]
  uint32_t* cand_idx;            // [max_tracks] track index, in cell order
  float4* cand_a;                // [max_tracks] (y, z_rel, sin phi, q/pT), in cell order
  float2* cand_b;                // [max_tracks] (time_ref, seed as bits), in cell order
  unsigned long long* out_key;   // [max_tracks] (d2 bits << 32 | seed of B) of out[A]; all ones = none
  int32_t* out_b;                // [max_tracks]
  unsigned long long* in_key;    // [max_tracks] (d2 bits << 32 | seed of A) of in[B]; all ones = none
};

__device__ __forceinline__ int merge_n(const MergeTracks& T, const MergeConsts& c) { return min(*T.n_tracks, c.max_tracks); }

// State part of the C5 transport (same statements, same order as tracklet.cuh::transport).
__device__ __forceinline__ bool merge_transport(float& x, float& y, float& z, float& s, float t, float k, float xn, float cB, float spm) {
  const float dx = xn - x;
  const float kc = cB * k;
  const float sn = s + kc * dx;
  if (!(fabsf(s) < spm && fabsf(sn) < spm)) return false;
  const float c = sqrtf(1.0f - s * s);
  const float cn = sqrtf(1.0f - sn * sn);
  const float ss = s + sn;
  const float cc = c + cn;
  const float icc = 1.0f / cc;
  const float T = ss * icc;
  const float q = 1.0f + T * T;
  const float rq = sqrtf(q);
  const float u = kc * dx;
  const float a = (u * u) * q;
  const float dS = (dx * rq) * (1.0f + a * (0.041666668f + a * (0.0046875f + a * 0.00069754466f)));
  y = y + dx * T;
  z = z + t * dS;
  s = sn;
  x = xn;
  return true;
}

__device__ __forceinline__ int merge_time_cell(float t, const MergeConsts& c) {
  return min(max(__float2int_rd(t * c.inv_cell), 0), c.n_tcell - 1);
}

// Row the state of a track sits on (reading M5) and its cell.
__global__ void __launch_bounds__(256) k_merge_cell_count(MergeTracks T, MergeScratch S, const __grid_constant__ MergeConsts c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= merge_n(T, c)) return;
  int rb = (int)floorf((T.x[i] - c.x0) / c.pitch + 0.5f);
  if (rb < 0 || rb >= c.n_rows || rb > T.first_row[i]) { S.cell_of[i] = 0xFFFFFFFFu; return; }   // reading M7: only a state at the inner end of its track is a candidate B
  const float tb = T.time_ref[i] + T.z[i] * c.inv_Z;
  const int sec = min(max(T.sector[i], 0), c.n_sectors - 1);
  const uint32_t cell = (uint32_t)((sec * c.n_rows + rb) * c.n_tcell + merge_time_cell(tb, c));
  S.cell_of[i] = cell;
  atomicAdd(S.cell_start + cell, 1u);
}

__global__ void __launch_bounds__(256) k_merge_cell_fill(MergeTracks T, MergeScratch S, const __grid_constant__ MergeConsts c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= merge_n(T, c)) return;
  const uint32_t cell = S.cell_of[i];
  if (cell == 0xFFFFFFFFu) return;
  const uint32_t pos = S.cell_start[cell] + atomicAdd(S.cell_cursor + cell, 1u);    // order inside a cell is irrelevant (ties are decided on seeds)
  S.cand_idx[pos] = (uint32_t)i;
  S.cand_a[pos] = make_float4(T.y[i], T.z[i], T.s[i], T.k[i]);
  S.cand_b[pos] = make_float2(T.time_ref[i], __int_as_float(T.seed[i]));
}

__global__ void __launch_bounds__(kMergeThreads) k_merge_match(MergeTracks T, MergeScratch S, const __grid_constant__ MergeConsts c) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= merge_n(T, c)) return;
  unsigned long long best = ~0ull;
  int best_b = -1;
  if (c.n_sectors >= 18) {
    const float ax = T.x[a], ay = T.y[a], az = T.z[a], as = T.s[a], at = T.t[a], ak = T.k[a], atr = T.time_ref[a];
    const uint32_t aseed = (uint32_t)T.seed[a];
    const int sec = T.sector[a], side = sec / 18, phi = sec % 18;
    const int fa = T.first_row[a], la = T.last_row[a];
    const int ra = (int)floorf((ax - c.x0) / c.pitch + 0.5f);            // row A's own state sits on
    const int r_lo = max(la + 1 - c.overlap, max(fa, ra) + 1), r_hi = min(la + 1 + c.gap, c.n_rows - 1);
    const float cs = sqrtf(1.0f - as * as);
    for (int isg = 0; isg < 2; ++isg) {
      const float sg = isg == 0 ? 1.0f : -1.0f;
      const int nb = side * 18 + (phi + (isg == 0 ? 1 : 17)) % 18;
      if (nb >= c.n_sectors) continue;
      const float x1 = ax * c.Cd + sg * (ay * c.Sd);
      const float y1 = ay * c.Cd - sg * (ax * c.Sd);
      const float s1 = as * c.Cd - sg * (cs * c.Sd);
      if (!(fabsf(s1) < c.sin_phi_max)) continue;
      for (int rb = r_lo; rb <= r_hi; ++rb) {
        float x2 = x1, y2 = y1, z2 = az, s2 = s1;
        if (!merge_transport(x2, y2, z2, s2, at, ak, __ldg(c.xr + rb), c.cB, c.sin_phi_max)) continue;
        const float tpred = atr + z2 * c.inv_Z;
        const uint32_t base = (uint32_t)((nb * c.n_rows + rb) * c.n_tcell);
        const uint32_t lo = __ldg(S.cell_start + base + merge_time_cell(tpred - c.t_window, c));
        const uint32_t hi = __ldg(S.cell_start + base + merge_time_cell(tpred + c.t_window, c) + 1);
        for (uint32_t q = lo; q < hi; ++q) {
          const float4 ca = S.cand_a[q];
          const float2 cb = S.cand_b[q];
          const float dy = y2 - ca.x;
          const float dz = (z2 - ca.y) + (atr - cb.x) * c.Z;
          const float ds = s2 - ca.z;
          const float dk = ak - ca.w;
          if (!(fabsf(dy) < c.cut_y && fabsf(dz) < c.cut_z && fabsf(ds) < c.cut_s && fabsf(dk) < c.cut_k)) continue;
          const float d2 = (dy * dy) * c.wy + (dz * dz) * c.wz + (ds * ds) * c.ws + (dk * dk) * c.wk;
          const unsigned long long hi_bits = (unsigned long long)__float_as_uint(d2) << 32;
          const unsigned long long key_b = hi_bits | (unsigned long long)(uint32_t)__float_as_int(cb.y);
          if (key_b < best) { best = key_b; best_b = (int)S.cand_idx[q]; }
          atomicMin(S.in_key + S.cand_idx[q], hi_bits | (unsigned long long)aseed);
        }
      }
    }
  }
  S.out_key[a] = best;
  S.out_b[a] = best_b;
}

// next / prev are pre-set to -1; *n_links to 0.
__global__ void __launch_bounds__(256) k_merge_link(MergeTracks T, MergeScratch S, int32_t* __restrict__ next, int32_t* __restrict__ prev,
                                                    int32_t* __restrict__ n_links, const __grid_constant__ MergeConsts c) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  bool linked = false;
  if (a < merge_n(T, c)) {
    const int b = S.out_b[a];
    if (b >= 0) {
      const unsigned long long key_a = (S.out_key[a] & 0xFFFFFFFF00000000ull) | (unsigned long long)(uint32_t)T.seed[a];
      if (S.in_key[b] == key_a) { next[a] = b; prev[b] = a; linked = true; }
    }
  }
  const unsigned m = __ballot_sync(0xffffffffu, linked);
  if (lane_id() == 0 && m) atomicAdd(n_links, __popc(m));
}

__global__ void __launch_bounds__(256) k_merge_root(MergeTracks T, const int32_t* __restrict__ prev, int32_t* __restrict__ root,
                                                    const __grid_constant__ MergeConsts c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= merge_n(T, c)) return;
  int r = i;
  int steps = 0;
  for (int p = prev[r]; p >= 0 && steps < c.n_rows; p = prev[r], ++steps) r = p;      // state rows strictly increase along a chain (M7): no cycles, <= n_rows pieces
  root[i] = r;
}

// ---- C10: merging across the central electrode (DESIGN.md §3 "C10", readings CE1..CE6) ----
// A track that approaches the electrode (dz/ds > 0 in the time-derived coordinate) continues in the mirror sector
// (S + 18) mod 36 of the other side with x, y, sin phi, q/pT unchanged and the time coordinate reflected.  Same binning,
// same row window, same reciprocal best match as C7; the state of A is carried to its last row and from there to the row
// of the candidate, which bounds where the crossing can be.
struct MergeCeConsts { float cut_t, wt; };

__global__ void __launch_bounds__(kMergeThreads) k_merge_ce_match(MergeTracks T, MergeScratch S, float* __restrict__ out_t,
                                                                   const __grid_constant__ MergeConsts c, const MergeCeConsts ce) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= merge_n(T, c)) return;
  unsigned long long best = ~0ull;
  int best_b = -1;
  float best_t = 0.0f;
  const float at = T.t[a];
  if (c.n_sectors == 36 && at > 0.0f) {                // CE2: only a track approaching the electrode can cross it
    const float ak = T.k[a], atr = T.time_ref[a];
    const uint32_t aseed = (uint32_t)T.seed[a];
    const int sec = T.sector[a], nb = (sec + 18) % 36;
    const int fa = T.first_row[a], la = T.last_row[a];
    float lx = T.x[a], ly = T.y[a], lz = T.z[a], ls = T.s[a];
    const int ra = (int)floorf((lx - c.x0) / c.pitch + 0.5f);
    const int r_lo = max(la + 1 - c.overlap, max(fa, ra) + 1), r_hi = min(la + 1 + c.gap, c.n_rows - 1);
    if (la >= 0 && la < c.n_rows && merge_transport(lx, ly, lz, ls, at, ak, __ldg(c.xr + la), c.cB, c.sin_phi_max)) {
      for (int rb = r_lo; rb <= r_hi; ++rb) {
        float x2 = lx, y2 = ly, z2 = lz, s2 = ls;
        if (!merge_transport(x2, y2, z2, s2, at, ak, __ldg(c.xr + rb), c.cB, c.sin_phi_max)) continue;
        const float zg = z2 - lz;
        const float hi = zg > 0.0f ? zg + zg : 0.0f;
        const float tpred = atr + z2 * c.inv_Z;        // A extrapolated through the electrode; B lies up to (hi + cut) / Z EARLIER
        const uint32_t base = (uint32_t)((nb * c.n_rows + rb) * c.n_tcell);
        const uint32_t lo = __ldg(S.cell_start + base + merge_time_cell(tpred - (hi + c.cut_z) * c.inv_Z - 0.5f, c));
        const uint32_t hi_q = __ldg(S.cell_start + base + merge_time_cell(tpred + c.t_window, c) + 1);
        for (uint32_t q = lo; q < hi_q; ++q) {
          const float4 ca = S.cand_a[q];               // (y, z_rel, sin phi, q/pT)
          const float2 cb = S.cand_b[q];               // (time_ref, seed)
          const float bt = T.t[S.cand_idx[q]];
          const float dy = y2 - ca.x;
          const float ds = s2 - ca.z;
          const float dk = ak - ca.w;
          const float dt = at + bt;
          const float dzm = (z2 - ca.y) + (atr - cb.x) * c.Z;
          const float ez = dzm < 0.0f ? dzm : (dzm > hi ? dzm - hi : 0.0f);
          if (!(fabsf(dy) < c.cut_y && fabsf(ez) < c.cut_z && fabsf(ds) < c.cut_s && fabsf(dk) < c.cut_k && fabsf(dt) < ce.cut_t)) continue;
          const float d2 = (dy * dy) * c.wy + (ez * ez) * c.wz + (ds * ds) * c.ws + (dk * dk) * c.wk + (dt * dt) * ce.wt;
          const unsigned long long hi_bits = (unsigned long long)__float_as_uint(d2) << 32;
          const unsigned long long key_b = hi_bits | (unsigned long long)(uint32_t)__float_as_int(cb.y);
          if (key_b < best) {
            best = key_b; best_b = (int)S.cand_idx[q];
            const float cl = fminf(fmaxf(dzm, 0.0f), hi);
            best_t = cb.x + (ca.y + 0.5f * cl) / c.Z;
          }
          atomicMin(S.in_key + S.cand_idx[q], hi_bits | (unsigned long long)aseed);
        }
      }
    }
  }
  S.out_key[a] = best;
  S.out_b[a] = best_b;
  out_t[a] = best_t;
}

// next / prev are pre-set to -1, t_ce to 0, *n_links to 0.
__global__ void __launch_bounds__(256) k_merge_ce_link(MergeTracks T, MergeScratch S, const float* __restrict__ out_t, int32_t* __restrict__ next,
                                                       int32_t* __restrict__ prev, float* __restrict__ t_ce, int32_t* __restrict__ n_links,
                                                       const __grid_constant__ MergeConsts c) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  bool linked = false;
  if (a < merge_n(T, c)) {
    const int b = S.out_b[a];
    if (b >= 0) {
      const unsigned long long key_a = (S.out_key[a] & 0xFFFFFFFF00000000ull) | (unsigned long long)(uint32_t)T.seed[a];
      if (S.in_key[b] == key_a) { next[a] = b; prev[b] = a; t_ce[a] = out_t[a]; linked = true; }
    }
  }
  const unsigned m = __ballot_sync(0xffffffffu, linked);
  if (lane_id() == 0 && m) atomicAdd(n_links, __popc(m));
}

// ---- C8: refit of the chains linked by C7 (DESIGN.md §3 "C8", readings F1..F6) ----
// One Kalman pass per chain of >= 2 pieces, from the outermost hit of the outermost piece inward to the innermost hit
// of the root piece, over the hits each piece owns, each piece in its own sector frame; state and covariance are
// rotated at every boundary.  transport / kalman_update are the constructor's (tracklet.cuh): same statements, same order.
struct RefitIo {
  const float2* hit_yt; const uint8_t* hit_row;   // (y, time) and pad row of every track hit, in hit_index order (tpc_tracks_t)
  const int32_t *n_hits; const int64_t* hit_offset; int64_t max_track_hits;
  const int32_t *next, *prev;               // C7 links
  int32_t *ok, *chain_hits, *chain_pieces;  // [max_tracks]
  float *rpar, *rcov;                       // [max_tracks * 7], [max_tracks * 9]
};

// Pass-through values for every track + the list of chain roots (order irrelevant: results are indexed by track).
__global__ void __launch_bounds__(256) k_refit_roots(MergeTracks T, RefitIo io, uint32_t* __restrict__ root_list, uint32_t* __restrict__ n_roots,
                                                     const __grid_constant__ MergeConsts c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  bool is_root = false;
  if (i < merge_n(T, c)) {
    is_root = io.prev[i] < 0 && io.next[i] >= 0;
    io.ok[i] = 0; io.chain_hits[i] = io.n_hits[i]; io.chain_pieces[i] = 1;
    float* rp = io.rpar + 7 * (size_t)i;
    rp[0] = T.x[i]; rp[1] = T.y[i]; rp[2] = T.z[i]; rp[3] = T.s[i]; rp[4] = T.t[i]; rp[5] = T.k[i]; rp[6] = T.time_ref[i];
    float* rc = io.rcov + 9 * (size_t)i;
#pragma unroll
    for (int k = 0; k < 9; ++k) rc[k] = 0.0f;
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

// Persistent warps, one lane per chain at a time, lanes refilled from a global counter once kRefitRefill of them are idle
// (chains are 60 .. 450 hits long: without the refill a warp waits for its longest chain).  One loop iteration = one hit:
// transport to its row, update; the next hit's (row, pad, time) are gathered one iteration ahead.
constexpr int kRefitRefill = 4;
__global__ void __launch_bounds__(kMergeThreads) k_refit_chains(MergeTracks T, RefitIo io, const uint32_t* __restrict__ root_list,
                                                                 const uint32_t* __restrict__ n_roots, uint32_t* __restrict__ work_counter,
                                                                 const __grid_constant__ MergeConsts c, const __grid_constant__ Consts tc) {
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
  TrackState S;
  S.x = S.y = S.z = S.s = S.t = S.k = 0.0f; S.c0 = S.c1 = S.c2 = S.c3 = S.c4 = S.c5 = 0.0f; S.d0 = S.d1 = S.d2 = 0.0f;
  for (;;) {
    const unsigned idle = __ballot_sync(0xffffffffu, !active && !exhausted);
    const unsigned busy = __ballot_sync(0xffffffffu, active);
    if (idle && (__popc(idle) >= kRefitRefill || busy == 0)) {
      if (!active && !exhausted) {
        const uint32_t e = (uint32_t)take_tracklets(work_counter, idle, lane);
        if (e >= n_work) {
          exhausted = true;
        } else {
          root = (int)root_list[e];
          int pm = root, pieces = 1, total = io.n_hits[root];
          bool complete = io.hit_offset[root] + io.n_hits[root] <= io.max_track_hits;      // hit list not cut by TPC_STATUS_TRACK_HIT_OVERFLOW
          for (int q = io.next[pm]; q >= 0; q = io.next[pm]) {
            if (pieces >= c.n_rows) { complete = false; break; }          // cannot happen (M7); never walk a corrupted link list for ever
            pm = q; ++pieces; total += io.n_hits[q];
            complete = complete && io.hit_offset[q] + io.n_hits[q] <= io.max_track_hits;
          }
          io.chain_hits[root] = total;
          io.chain_pieces[root] = pieces;
          if (!complete) io.ok[root] = -1;
          S.x = T.x[pm]; S.y = T.y[pm]; S.z = T.z[pm]; S.s = T.s[pm]; S.t = T.t[pm]; S.k = T.k[pm];
          S.c0 = S.c1 = S.c2 = S.c3 = S.c4 = S.c5 = 0.0f; S.d0 = S.d1 = S.d2 = 0.0f;
          p = pm; off = io.hit_offset[pm]; j = off + io.n_hits[pm] - 1; tref = T.time_ref[pm];
          if (complete) { hy = io.hit_yt[j]; hr = io.hit_row[j]; } else { hr = 0; }
          const bool ok0 = transport(S, xr[hr], tc.cB, tc.sin_phi_max);       // to the outermost hit, then the reset covariance
          S.c0 = tc.c0_y2; S.c1 = 0.0f; S.c2 = tc.c0_s2; S.c3 = 0.0f; S.c4 = 0.0f; S.c5 = tc.c0_k2; S.d0 = tc.c0_z2; S.d1 = 0.0f; S.d2 = tc.c0_t2;
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
      bool good = transport(S, xr[hr], tc.cB, tc.sin_phi_max);
      if (good) {
        kalman_update(S, hy.x, (hy.y - tref) * tc.Z, tc.ry, tc.rz);
        if (j > off) {
          --j; hy = ny; hr = nr;
        } else if (p == root) {                        // innermost hit of the root piece: done
          io.ok[root] = 1;
          float* rp = io.rpar + 7 * (size_t)root;
          rp[0] = S.x; rp[1] = S.y; rp[2] = S.z; rp[3] = S.s; rp[4] = S.t; rp[5] = S.k;      // rp[6] = time_ref of the root: already there
          float* rc = io.rcov + 9 * (size_t)root;
          rc[0] = S.c0; rc[1] = S.c1; rc[2] = S.c2; rc[3] = S.c3; rc[4] = S.c4; rc[5] = S.c5; rc[6] = S.d0; rc[7] = S.d1; rc[8] = S.d2;
          active = false;
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
            S.c1 = S.c1 * J; S.c2 = (S.c2 * J) * J; S.c4 = S.c4 * J;
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

// ---- C9: time and offset at which a track passes the beam line (DESIGN.md §3 "C9") ----
// One thread per state: transport to x = 0 (the beam axis in every sector frame); vertex_time = time_ref + z / Z.
__global__ void __launch_bounds__(256) k_vertex_time(const int32_t* __restrict__ n_tracks, int max_tracks, const float* __restrict__ par7,
                                                     int32_t* __restrict__ ok, float* __restrict__ vertex_time, float* __restrict__ vertex_y,
                                                     float Z, float cB, float sin_phi_max) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= min(*n_tracks, max_tracks)) return;
  const float* q = par7 + 7 * (size_t)i;
  float x = q[0], y = q[1], z = q[2], s = q[3];
  const bool good = merge_transport(x, y, z, s, q[4], q[5], 0.0f, cB, sin_phi_max);
  ok[i] = good ? 1 : 0;
  vertex_time[i] = good ? q[6] + z / Z : 0.0f;
  vertex_y[i] = good ? y : 0.0f;
}

}  // namespace tpc
