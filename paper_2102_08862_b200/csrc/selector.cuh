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

constexpr int kSelectorThreads = 256;   // 8 tracklets per CTA

__device__ __forceinline__ unsigned long long tracklet_key(int n_hits, uint32_t seed_orig) {
  return ((unsigned long long)(uint32_t)n_hits << 32) | (unsigned long long)(0xFFFFFFFFu - seed_orig);
}

__global__ void __launch_bounds__(kSelectorThreads) k_selector_claim(TrackletStore tl, const int32_t* __restrict__ counters,
                                                                     unsigned long long* __restrict__ claim,
                                                                     const __grid_constant__ Consts c) {
  const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j >= counters[0]) return;
  const int nh = tl.n_hits[j];
  if (nh < c.min_hits) return;
  const unsigned long long key = tracklet_key(nh, tl.seed_orig[j]);
  const int first = tl.first_row[j], last = tl.last_row[j];
  const int* rows = tl.row_hit + (size_t)j * kRowStride;
  for (int r = (first & ~31) + (int)lane_id(); r <= last; r += 32) {
    if (r < first) continue;
    const int m = rows[r];
    if (m >= 0) atomicMax(claim + m, key);
  }
}

// owned[j] = number of hits tracklet j still owns if that reaches min_hits, else 0; flag[j] = owned[j] > 0.
// Entries j >= n_tracklets are written as 0 so the scans can run over the whole capacity.
__global__ void __launch_bounds__(kSelectorThreads) k_selector_count(TrackletStore tl, const int32_t* __restrict__ counters,
                                                                     const unsigned long long* __restrict__ claim,
                                                                     uint32_t* __restrict__ owned, uint32_t* __restrict__ flag,
                                                                     int max_tracklets, const __grid_constant__ Consts c) {
  const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j >= max_tracklets) return;
  int n_owned = 0;
  if (j < counters[0]) {
    const int nh = tl.n_hits[j];
    if (nh >= c.min_hits) {
      const unsigned long long key = tracklet_key(nh, tl.seed_orig[j]);
      const int first = tl.first_row[j], last = tl.last_row[j];
      const int* rows = tl.row_hit + (size_t)j * kRowStride;
      for (int r = (first & ~31) + (int)lane_id(); r - (int)lane_id() <= last; r += 32) {
        bool mine = false;
        if (r >= first && r <= last) {
          const int m = rows[r];
          mine = m >= 0 && claim[m] == key;
        }
        n_owned += __popc(__ballot_sync(0xffffffffu, mine));
      }
    }
  }
  if (lane_id() == 0) {
    const bool keep = n_owned >= c.min_hits;
    owned[j] = keep ? (uint32_t)n_owned : 0u;
    flag[j] = keep ? 1u : 0u;
  }
}

struct TrackOutputs {   // device pointers of tpc_tracks_t (include/tpc_tracker.h)
  int32_t max_tracks; int64_t max_track_hits;
  int32_t* n_tracks; int64_t* n_track_hits; int32_t* status;
  int32_t *seed_hit, *sector, *first_row, *last_row, *n_hits; int64_t* hit_offset;
  float *x, *y, *z_rel, *time_ref, *sin_phi, *dzds, *q_pt, *cov9;
  int32_t* hit_index;
};

// track_idx / hit_off are the exclusive scans of flag / owned; their totals sit behind the last tile offset.
__global__ void __launch_bounds__(kSelectorThreads) k_selector_emit(
    TrackletStore tl, const int32_t* __restrict__ counters, const unsigned long long* __restrict__ claim,
    const uint32_t* __restrict__ flag_in, const uint32_t* __restrict__ track_idx, const uint32_t* __restrict__ hit_off,
    const uint32_t* __restrict__ track_total, const uint32_t* __restrict__ hit_total,
    const uint32_t* __restrict__ orig, const uint16_t* __restrict__ hsr, const uint32_t* __restrict__ start_hits,
    const uint32_t* __restrict__ n_invalid, TrackOutputs o, const __grid_constant__ Consts c) {
  const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (j == 0 && lane_id() == 0) {
    const uint32_t nt = *track_total, nh = *hit_total;
    *o.n_tracks = (int32_t)nt;
    *o.n_track_hits = (int64_t)nh;
    int st = 0;
    if (counters[1] > counters[0]) st |= 1;                 // TPC_STATUS_TRACKLET_OVERFLOW
    if ((int64_t)nt > (int64_t)o.max_tracks) st |= 2;       // TPC_STATUS_TRACK_OVERFLOW
    if ((int64_t)nh > o.max_track_hits) st |= 4;            // TPC_STATUS_TRACK_HIT_OVERFLOW
    if (*n_invalid) st |= 8;                                // TPC_STATUS_INVALID_CLUSTERS
    *o.status = st;
  }
  if (j >= counters[0]) return;
  // flag is re-derived from the scanned arrays' neighbours being unavailable for the last element -> use flag_in
  if (flag_in[j] == 0) return;
  const uint32_t ti = track_idx[j];
  const uint32_t off = hit_off[j];
  if ((int64_t)ti >= (int64_t)o.max_tracks) return;
  const int nh = tl.n_hits[j];
  const unsigned long long key = tracklet_key(nh, tl.seed_orig[j]);
  const int first = tl.first_row[j], last = tl.last_row[j];
  const int* rows = tl.row_hit + (size_t)j * kRowStride;
  int n_owned = 0, own_first = -1, own_last = -1;
  for (int r = (first & ~31) + (int)lane_id(); r - (int)lane_id() <= last; r += 32) {
    int m = -1;
    bool mine = false;
    if (r >= first && r <= last) {
      m = rows[r];
      mine = m >= 0 && claim[m] == key;
    }
    const unsigned b = __ballot_sync(0xffffffffu, mine);
    if (mine) {
      const int64_t pos = (int64_t)off + n_owned + __popc(b & ((1u << lane_id()) - 1u));
      if (pos < o.max_track_hits) o.hit_index[pos] = (int32_t)orig[m];
    }
    if (b) {
      const int base = r - (int)lane_id();
      if (own_first < 0) own_first = base + __ffs(b) - 1;
      own_last = base + 31 - __clz(b);
    }
    n_owned += __popc(b);
  }
  if (lane_id() == 0) {
    const size_t cap = tl.cap;
    o.seed_hit[ti] = (int32_t)tl.seed_orig[j];
    o.sector[ti] = (int32_t)(hsr[start_hits[j]] / c.n_rows);
    o.first_row[ti] = own_first;
    o.last_row[ti] = own_last;
    o.n_hits[ti] = n_owned;
    o.hit_offset[ti] = (int64_t)off;
    o.x[ti] = tl.par[0 * cap + j]; o.y[ti] = tl.par[1 * cap + j]; o.z_rel[ti] = tl.par[2 * cap + j];
    o.sin_phi[ti] = tl.par[3 * cap + j]; o.dzds[ti] = tl.par[4 * cap + j]; o.q_pt[ti] = tl.par[5 * cap + j];
    o.time_ref[ti] = tl.par[6 * cap + j];
    if (o.cov9) for (int i = 0; i < 9; ++i) o.cov9[(size_t)ti * 9 + i] = tl.cov[i * cap + j];
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
  const int first = tl.first_row[j], last = tl.last_row[j];
  const int* rows = tl.row_hit + (size_t)j * kRowStride;
  if (tap_row_hit)
    for (int r = lane_id(); r < c.n_rows; r += 32) {
      int v = -1;
      if (r >= first && r <= last) { const int m = rows[r]; if (m >= 0) v = (int32_t)orig[m]; }
      tap_row_hit[(size_t)j * c.n_rows + r] = v;
    }
  if (lane_id() == 0) {
    if (tap_seed) tap_seed[j] = (int32_t)tl.seed_orig[j];
    if (tap_n_hits) tap_n_hits[j] = tl.n_hits[j];
  }
  if (tap_par && lane_id() < 7) tap_par[(size_t)j * 7 + lane_id()] = tl.par[lane_id() * tl.cap + j];
}

}  // namespace tpc
