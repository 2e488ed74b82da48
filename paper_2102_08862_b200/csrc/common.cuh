// Device-side definitions shared by the tracker's kernels (sm_100a).  See DESIGN.md §4 (data layout).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpc {

constexpr int kRowStride = 160;          // padded row count of one tracklet's row->hit table (5 x 32 lanes)
constexpr uint32_t kInvalidRank = 0xFFFFFFFFu;

// Constants of one tracker handle, passed by value to every kernel.  All fp32 decision constants are derived
// on the host in double from the fp32 parameter values and rounded once ("Notation").
struct Consts {
  // geometry
  int n_rows, n_sr, n_tb, n_pb, n_bins;  // rows per sector, sector-rows, time bins and pad bins per sector-row, n_sr*n_tb*n_pb
  float max_time, inv_bin_w;             // validity bound of the time coordinate; 1 / grid bin width (time)
  float inv_n_rows;                      // (float)(1 / n_rows), for row = sector_row mod n_rows without a division
  float Z, inv_Z, P;                     // time-bin size [cm], its inverse (grid lookups only), pad pitch
  // neighbours finder (C2)
  float W1, Ay, Az, wy, wz, chi2_cut;
  float finder_tw, finder_yw;            // half widths of the grid lookup: time bins / cm, each with a safety margin
  // tracklet constructor (C5)
  float ry, rz, cB, sin_phi_max, win_slope, win_const;
  float c0_y2, c0_s2, c0_k2, c0_z2, c0_t2;
  int miss_limit, min_hits, seed_min_hits;
  // per-row tables in device memory owned by the handle
  const float* xr;                       // [n_rows] x of the pad row
  const float* cr;                       // [n_rows] pad centre 0.5*(n_pads-1)
  const int* npads;                      // [n_rows]
  const float* yoff;                     // [n_rows] half width of the row in cm: pad bin = floor((y + yoff) * pscale)
  const float* pscale;                   // [n_rows] n_pb / (row width in cm)
  const float4* rowtab;                  // [n_rows] (n_pads - 0.5, cr, yoff, pscale): one 16-byte load per cluster in the ingest
};

// Grid bin of a time value: monotone non-decreasing in t, so a lookup over [bin(t_lo), bin(t_hi)] is a
// superset of the hits with time in [t_lo, t_hi].  The grid only accelerates; every decision is re-made by
// the exact fp32 predicate on the candidates.
__device__ __forceinline__ int time_bin(float t, const Consts& c) {
  int b = __float2int_rd(t * c.inv_bin_w);         // = (int)floorf(.) in one instruction
  return min(max(b, 0), c.n_tb - 1);
}

// Grid pad bin of a local y in a row (yoff, pscale of that row): monotone non-decreasing in y for the same reason.
__device__ __forceinline__ int pad_bin(float y, float yoff, float pscale, const Consts& c) {
  int b = __float2int_rd((y + yoff) * pscale);
  return min(max(b, 0), c.n_pb - 1);
}

// Grid bin index.  Inside a sector-row the bins are TIME-MAJOR: ((sector_row * n_tb + time_bin) * n_pb + pad_bin), so
// that (a) all hits of a sector-row inside a time range are ONE contiguous span of the sorted hit arrays -- what a CTA
// stages into shared memory with one bulk copy -- and (b) the pad bins pb0..pb1 of one time bin are contiguous: a
// lookup window is one span per grid time bin it touches.
__device__ __forceinline__ uint32_t grid_bin(int sr, int tb, int pb, const Consts& c) {
  return (uint32_t)((sr * c.n_tb + tb) * c.n_pb + pb);
}

__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }

}  // namespace tpc
