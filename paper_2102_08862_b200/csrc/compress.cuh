// C11 track-based hit rejection and track-model residual coding (the step behind the path;
// "removal of TPC hits of tracks not used for physics, reduction of the hit property entropy" -- the reason the
// tracking runs online).  Definition: DESIGN.md §3 "C11", readings R11-1..R11-6:
//   * every hit owned by a track with |q/pT| > reject_qpt is rejected (flag by original cluster index); hits no track owns
//     are kept;
//   * the hits of every kept track are coded as residuals against a Kalman prediction that starts from the track's C6
//     parameters and covariance and is updated with the RECONSTRUCTED hit (prediction + symbol x step), so a decoder that
//     reads the same header and symbols runs the same filter: transport -> (qy, qz) = rintf(residual / step) -> update.
// transport / kalman_update are the constructor's (tracklet.cuh): same statements, same order -> symbols equal the oracle's.
// Work distribution as in k_refit_chains: persistent warps, one lane per track, lanes refilled from a counter.
#pragma once
#include "common.cuh"
#include "merge.cuh"
#include "tracklet.cuh"

namespace tpc {

struct CompressIo {
  const int32_t* n_tracks; int32_t max_tracks; int64_t max_track_hits;
  const int32_t* n_hits; const int64_t* hit_offset; const int32_t* hit_index;
  const float2* hit_yt; const uint8_t* hit_row;
  const float *x, *y, *z, *s, *t, *k, *time_ref, *cov9;
  uint8_t* reject; int32_t* ok; int16_t *qy, *qz;
  float reject_qpt, step_y, step_z;
};

// One warp per track: the rejection decision, the reject flags of a rejected track's hits, zeroed symbols for every hit that
// will not be coded.  ok: -1 rejected, 0 not coded (hit list cut by a capacity overflow; or set later: transport FAIL), 1 coded.
__global__ void __launch_bounds__(256) k_compress_reject(CompressIo io) {
  const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (k >= min(*io.n_tracks, io.max_tracks)) return;
  const bool rej = fabsf(io.k[k]) > io.reject_qpt;
  const int64_t off = io.hit_offset[k];
  const int nh = io.n_hits[k];
  const bool complete = off + nh <= io.max_track_hits;
  if (lane_id() == 0) io.ok[k] = rej ? -1 : (complete ? 1 : 0);
  if (rej || !complete)
    for (int64_t j = off + lane_id(); j < min(off + nh, io.max_track_hits); j += 32) {
      if (rej) io.reject[io.hit_index[j]] = 1;
      io.qy[j] = 0; io.qz[j] = 0;
    }
}

constexpr int kCompressRefill = 4;
__global__ void __launch_bounds__(kMergeThreads) k_compress_tracks(CompressIo io, uint32_t* __restrict__ work_counter, const __grid_constant__ Consts tc) {
  __shared__ float xr[kRowStride];
  for (int r = threadIdx.x; r < tc.n_rows; r += blockDim.x) xr[r] = tc.xr[r];
  __syncthreads();
  const uint32_t n_work = (uint32_t)min(*io.n_tracks, io.max_tracks);
  const unsigned lane = lane_id();
  bool active = false, exhausted = false;
  int k = -1;
  int64_t j = 0, j_end = 0;
  float tref = 0.0f;
  float2 hy = make_float2(0.0f, 0.0f);
  int hr = 0;
  TrackState S;
  S.x = S.y = S.z = S.s = S.t = S.k = 0.0f; S.c0 = S.c1 = S.c2 = S.c3 = S.c4 = S.c5 = 0.0f; S.d0 = S.d1 = S.d2 = 0.0f;
  for (;;) {
    const unsigned idle = __ballot_sync(0xffffffffu, !active && !exhausted);
    const unsigned busy = __ballot_sync(0xffffffffu, active);
    if (idle && (__popc(idle) >= kCompressRefill || busy == 0)) {
      if (!active && !exhausted) {
        const uint32_t e = (uint32_t)take_tracklets(work_counter, idle, lane);
        if (e >= n_work) {
          exhausted = true;
        } else if (io.ok[e] == 1) {                    // a kept track with a complete hit list
          k = (int)e;
          S.x = io.x[k]; S.y = io.y[k]; S.z = io.z[k]; S.s = io.s[k]; S.t = io.t[k]; S.k = io.k[k];
          const float* cv = io.cov9 + 9 * (size_t)k;
          S.c0 = cv[0]; S.c1 = cv[1]; S.c2 = cv[2]; S.c3 = cv[3]; S.c4 = cv[4]; S.c5 = cv[5]; S.d0 = cv[6]; S.d1 = cv[7]; S.d2 = cv[8];
          tref = io.time_ref[k];
          j = io.hit_offset[k]; j_end = j + io.n_hits[k];
          hy = io.hit_yt[j]; hr = io.hit_row[j];
          active = true;
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
      if (j + 1 < j_end) { ny = io.hit_yt[j + 1]; nr = io.hit_row[j + 1]; }          // the next hit, one iteration ahead
      if (transport(S, xr[hr], tc.cB, tc.sin_phi_max)) {
        const float ry = hy.x - S.y;
        const float rz = (hy.y - tref) * tc.Z - S.z;
        int iy = (int)rintf(ry / io.step_y), iz = (int)rintf(rz / io.step_z);
        iy = min(max(iy, -32767), 32767); iz = min(max(iz, -32767), 32767);
        io.qy[j] = (int16_t)iy; io.qz[j] = (int16_t)iz;
        const float yq = S.y + (float)iy * io.step_y, zq = S.z + (float)iz * io.step_z;      // what a decoder reconstructs
        kalman_update(S, yq, zq, tc.ry, tc.rz);
        ++j; hy = ny; hr = nr;
        if (j == j_end) active = false;
      } else {                                         // FAIL: not coded from here on
        io.ok[k] = 0;
        for (int64_t q = j; q < j_end; ++q) { io.qy[q] = 0; io.qz[q] = 0; }
        active = false;
      }
    }
  }
}

}  // namespace tpc
