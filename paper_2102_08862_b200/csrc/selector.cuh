// C6 tracklet selector (BASELINE.json L5 item 5: "resolves shared hits by an atomicMax claim on the key
// (nHits, -id)").  One warp per tracklet, lanes over rows (the row->hit table is tracklet-major, 160 ints):
//   claim : claim[hit] = max(claim[hit], key)       key = nHits << 32 | (0xFFFFFFFF - id), id = orig(start hit)
//   count : owned = #hits with claim[hit] == key;   a track is emitted iff owned >= min_hits
//   scan  : track index / hit offset = exclusive scans of the flags / owned counts  (deterministic order)
//   emit  : track record + its owned hits (original indices, ascending row), parameters unchanged (no refit)
// One pass, no re-claiming after a tracklet is dropped (DESIGN.md §3 C6).
#pragma once
#include "common.cuh"
#include "tracklet.cuh"

namespace tpc {

#ifndef TPC_SELECTOR_THREADS
#define TPC_SELECTOR_THREADS 256
#endif
constexpr int kSelectorThreads = TPC_SELECTOR_THREADS;   // 8 tracklets per CTA at 256

// Claim, step 1: every tracklet claims its TOP hit (one thread per tracklet).  The ~7 tracklets that follow one track from its
// different seed chains nearly always end on the same hit, so afterwards claim[top hit] names the best of them (or an even
// better tracklet through that hit): the LEADER step 2 compares against.
__global__ void __launch_bounds__(256) k_selector_claim_top(TrackletStore tl, const int32_t* __restrict__ counters,
                                                            unsigned long long* __restrict__ claim, const __grid_constant__ Consts c) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= counters[0]) return;
  const int4 meta = tl.meta[j];                      // n_hits, first_row, last_row, seed_orig
  if (meta.x < c.min_hits) return;
  const int top = tl.row_hit[(size_t)j * kRowStride + meta.z];
  if (top >= 0) atomicMax(claim + top, tracklet_key(meta.x, (uint32_t)meta.w, (uint32_t)j));
}

// Claim, step 2: one warp per tracklet, lanes over rows.  L = the tracklet named by claim[top hit]: its key is >= this one's
// and it holds the top hit.  If L is another tracklet, every hit this tracklet shares with L ON THE SAME ROW needs no atomic:
// L's key is larger, and L either claims that hit itself or skips it for the same reason against a still larger key -- the
// chain of leaders is strictly increasing in the key, so it ends at a tracklet that does claim the hit.  claim[] therefore
// ends as the same maximum over all tracklets (whatever value the racing read of claim[top] returns: any tracklet it can name
// qualifies), with ~ 6 of 7 atomics replaced by a coalesced read of the leader's row table.
// (Claiming from inside the constructor when a tracklet retires was measured: it stalls the whole warp on the row
// reads and costs 10 ms against 6 ms for a claim kernel.)
__global__ void __launch_bounds__(kSelectorThreads) k_selector_claim(TrackletStore tl, const int32_t* __restrict__ counters,
                                                                     unsigned long long* __restrict__ claim,
                                                                     const __grid_constant__ Consts c) {
  constexpr int kWords = kRowStride / 32;
  const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j >= counters[0]) return;
  const int4 meta = tl.meta[j];                      // n_hits, first_row, last_row, seed_orig
  const int nh = meta.x;
  if (nh < c.min_hits) return;
  const unsigned long long key = tracklet_key(nh, (uint32_t)meta.w, (uint32_t)j);
  const int first = meta.y, last = meta.z;
  const int* rows = tl.row_hit + (size_t)j * kRowStride;
  int m[kWords];
#pragma unroll
  for (int i = 0; i < kWords; ++i) {
    const int r = i * 32 + (int)lane_id();
    m[i] = (r >= first && r <= last) ? rows[r] : -1;
  }
  const int top = rows[last];
  int L = j;
  if (top >= 0) L = (int)(claim[top] & ((1ull << kKeySlotBits) - 1ull));
  if (L != j) {
    const int4 ml = tl.meta[L];
    const int* rows_l = tl.row_hit + (size_t)L * kRowStride;
#pragma unroll
    for (int i = 0; i < kWords; ++i) {
      const int r = i * 32 + (int)lane_id();
      const int h = (r >= ml.y && r <= ml.z) ? rows_l[r] : -1;
      if (h == m[i]) m[i] = -1;                       // shared with the leader on this row: the leader's claim covers it
    }
  }
#pragma unroll
  for (int i = 0; i < kWords; ++i)
    if (m[i] >= 0) atomicMax(claim + m[i], key);
}


// Count step, over the HITS: claim[h] names the tracklet slot that owns hit h (low bits of the key), so one coalesced pass
// over the claim array and one 32-bit atomicAdd per claimed hit (the counters of 1.2e7 slots stay in L2) replace a second
// gather of every tracklet's claims (7e8 scattered 8-byte reads: 4.4 ms against 1.6 ms on configs[3]).  owned_raw is zeroed
// before.
__global__ void __launch_bounds__(256) k_selector_count_hits(const unsigned long long* __restrict__ claim, const uint32_t* __restrict__ bin_start,
                                                             uint32_t* __restrict__ owned_raw, const __grid_constant__ Consts c) {
  const uint32_t n_valid = __ldg(bin_start + c.n_bins);
  const uint32_t h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_valid) return;
  const unsigned long long cl = claim[h];
  if (cl) atomicAdd(owned_raw + (uint32_t)(cl & ((1ull << kKeySlotBits) - 1ull)), 1u);
}

// owned[j] = number of hits tracklet j still owns if that reaches min_hits, else 0 (in place); flag[j] = owned[j] > 0.
// Runs over the whole capacity (slots >= n_tracklets hold 0) so that the scans can, too.
__global__ void __launch_bounds__(256) k_selector_flag(uint32_t* __restrict__ owned, uint32_t* __restrict__ flag, int max_tracklets,
                                                       const __grid_constant__ Consts c) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= max_tracklets) return;
  const uint32_t n = owned[j];
  const bool keep = n >= (uint32_t)c.min_hits;
  if (!keep && n) owned[j] = 0u;
  flag[j] = keep ? 1u : 0u;
}

struct TrackOutputs {   // device pointers of tpc_tracks_t (include/tpc_tracker.h)
  int32_t max_tracks; int64_t max_track_hits;
  int32_t* n_tracks; int64_t* n_track_hits; int32_t* status;
  int32_t *seed_hit, *sector, *first_row, *last_row, *n_hits; int64_t* hit_offset;
  float *x, *y, *z_rel, *time_ref, *sin_phi, *dzds, *q_pt, *cov9;
  int32_t* hit_index;
  float2* hit_yt; uint8_t* hit_row;   // optional (NULL = not wanted)
};

// track_slot[track_idx[j]] = j for every tracklet that became a track: the emit kernel then runs one warp per TRACK
// (1.8e6 in configs[3]) instead of one per tracklet slot (1.2e7, most of which had nothing to emit).
__global__ void __launch_bounds__(256) k_selector_map(const int32_t* __restrict__ counters, const uint32_t* __restrict__ flag,
                                                      const uint32_t* __restrict__ track_idx, uint32_t* __restrict__ track_slot) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j < counters[0] && flag[j]) track_slot[track_idx[j]] = (uint32_t)j;
}

// One warp per track.  track_idx / hit_off are the exclusive scans of flag / owned; their totals sit behind the last
// tile offset.
__global__ void __launch_bounds__(kSelectorThreads) k_selector_emit(
    TrackletStore tl, const int32_t* __restrict__ counters, const unsigned long long* __restrict__ claim,
    const uint32_t* __restrict__ track_slot, const uint32_t* __restrict__ hit_off,
    const uint32_t* __restrict__ track_total, const uint32_t* __restrict__ hit_total,
    const uint32_t* __restrict__ orig, const float2* __restrict__ yt, const uint16_t* __restrict__ hsr, const uint32_t* __restrict__ start_hits,
    const uint32_t* __restrict__ n_invalid, TrackOutputs o, const __grid_constant__ Consts c) {
  constexpr int kWords = kRowStride / 32;
  const uint32_t ti = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const uint32_t nt = *track_total;
  if (ti == 0 && lane_id() == 0) {
    const uint32_t nh = *hit_total;
    *o.n_tracks = (int32_t)nt;
    *o.n_track_hits = (int64_t)nh;
    int st = 0;
    if (counters[1] > counters[0]) st |= 1;                 // TPC_STATUS_TRACKLET_OVERFLOW
    if ((int64_t)nt > (int64_t)o.max_tracks) st |= 2;       // TPC_STATUS_TRACK_OVERFLOW
    if ((int64_t)nh > o.max_track_hits) st |= 4;            // TPC_STATUS_TRACK_HIT_OVERFLOW
    if (*n_invalid) st |= 8;                                // TPC_STATUS_INVALID_CLUSTERS
    *o.status = st;
  }
  if (ti >= nt || (int64_t)ti >= (int64_t)o.max_tracks) return;
  const int j = (int)track_slot[ti];
  const uint32_t off = hit_off[j];
  const int* rows = tl.row_hit + (size_t)j * kRowStride;
  const int4 meta = tl.meta[j];                      // n_hits, first_row, last_row, seed_orig
  const unsigned long long key = tracklet_key(meta.x, (uint32_t)meta.w, (uint32_t)j);
  int mrow[kWords];
  unsigned long long cl[kWords];
#pragma unroll
  for (int i = 0; i < kWords; ++i) {                 // the five row words, then the five claim gathers, back to back
    const int r = i * 32 + (int)lane_id();
    mrow[i] = (r >= meta.y && r <= meta.z) ? rows[r] : -1;
  }
#pragma unroll
  for (int i = 0; i < kWords; ++i) cl[i] = mrow[i] >= 0 ? claim[mrow[i]] : 0ull;
  int n_owned = 0, own_first = -1, own_last = -1;
#pragma unroll
  for (int i = 0; i < kWords; ++i) {
    const unsigned b = __ballot_sync(0xffffffffu, mrow[i] >= 0 && cl[i] == key);      // the rows this tracklet still owns
    if (b >> lane_id() & 1u) {
      const int m = mrow[i];
      const int64_t pos = (int64_t)off + n_owned + __popc(b & ((1u << lane_id()) - 1u));
      if (pos < o.max_track_hits) {
        o.hit_index[pos] = (int32_t)orig[m];
        if (o.hit_yt) o.hit_yt[pos] = yt[m];
        if (o.hit_row) o.hit_row[pos] = (uint8_t)(i * 32 + (int)lane_id());
      }
    }
    if (b) {
      if (own_first < 0) own_first = i * 32 + __ffs(b) - 1;
      own_last = i * 32 + 31 - __clz(b);
    }
    n_owned += __popc(b);
  }
  if (lane_id() == 0) {
    const float4* rec = tl.rec + 4 * (size_t)j;
    const float4 q0 = rec[0], q1 = rec[1], q2 = rec[2], q3 = rec[3];
    o.seed_hit[ti] = meta.w;
    o.sector[ti] = (int32_t)(hsr[start_hits[j]] / c.n_rows);
    o.first_row[ti] = own_first;
    o.last_row[ti] = own_last;
    o.n_hits[ti] = n_owned;
    o.hit_offset[ti] = (int64_t)off;
    o.x[ti] = q0.x; o.y[ti] = q0.y; o.z_rel[ti] = q0.z; o.sin_phi[ti] = q0.w; o.dzds[ti] = q1.x; o.q_pt[ti] = q1.y;
    o.time_ref[ti] = q3.w;
    if (o.cov9) {
      float* cv = o.cov9 + (size_t)ti * 9;
      cv[0] = q1.z; cv[1] = q1.w; cv[2] = q2.x; cv[3] = q2.y; cv[4] = q2.z; cv[5] = q2.w; cv[6] = q3.x; cv[7] = q3.y; cv[8] = q3.z;
    }
  }
}

// Parity taps of the tracklets (by original cluster index); one warp per tracklet slot.
__global__ void __launch_bounds__(kSelectorThreads) k_export_tracklets(
    TrackletStore tl, const int32_t* __restrict__ counters, const uint32_t* __restrict__ orig,
    int32_t* __restrict__ tap_n, int32_t* __restrict__ tap_seed, int32_t* __restrict__ tap_n_hits,
    int32_t* __restrict__ tap_row_hit, float* __restrict__ tap_par, int tap_capacity, const __grid_constant__ Consts c) {
  const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j == 0 && lane_id() == 0 && tap_n) *tap_n = counters[0];
  if (j >= counters[0] || j >= tap_capacity) return;
  const int4 meta = tl.meta[j];
  const int first = meta.y, last = meta.z;
  const int* rows = tl.row_hit + (size_t)j * kRowStride;
  if (tap_row_hit)
    for (int r = lane_id(); r < c.n_rows; r += 32) {
      int v = -1;
      if (r >= first && r <= last) { const int m = rows[r]; if (m >= 0) v = (int32_t)orig[m]; }
      tap_row_hit[(size_t)j * c.n_rows + r] = v;
    }
  if (lane_id() == 0) {
    if (tap_seed) tap_seed[j] = meta.w;
    if (tap_n_hits) tap_n_hits[j] = meta.x;
  }
  if (tap_par && lane_id() < 7) {                     // x, y, z_rel, sin_phi, dzds, q_pt, time_ref
    const float* rec = reinterpret_cast<const float*>(tl.rec + 4 * (size_t)j);
    tap_par[(size_t)j * 7 + lane_id()] = rec[lane_id() < 6 ? lane_id() : 15];
  }
}

}  // namespace tpc
