// C0 TPC cluster finder (the step in front of the tracking path; clusterization is
// part of the synchronous GPU load; zero suppression happens in the readout).  Definition: DESIGN.md §3 "C0",
// readings D1..D6 -- a sample is a PEAK iff its ADC reaches the threshold and it beats its (up to) 8 neighbours in
// (pad, time) of the same sector-row (larger ADC, ties to the earlier sample); the cluster of a peak is the centre of
// gravity of its 3 x 3 window, summed in fp32 in the stated order.
//
// Input: samples sorted by (sector_row, time bin, pad).  A GROUP = the samples of one (sector_row, time bin), contiguous
// and pad-sorted, so
//   * the neighbours in the same time bin are the samples at i - 1 / i + 1 (if their pad differs by one),
//   * the time bin before / after is the group before / after (if it has the same sector_row and time +- 1), where the
//     pads p-1, p, p+1 are at most three consecutive entries found by a short binary search.
//
// Shape (round 2, second version): ONE pass over the samples with everything a window needs in shared memory.  A CTA owns a
// tile of kCfTile consecutive samples and stages them plus kCfHalo samples on either side (the group before the first sample's
// group and the group after the last one's lie inside the halo: a group holds at most one sample per pad).  In shared memory:
// head flags -> block-wide running maximum = start of every sample's group -> end of every group; then one sample per thread
// and round: decision and the three sums from shared memory only; ordered compaction of the round's peaks (ballot + the
// eight warp counts) into a staging area at the tile's own offset.  A scan over the per-tile counts and a copy of the staged clusters
// to their final place finish the job (deterministic order, no atomics).  A sample whose groups are not completely inside the
// staged window (only possible with more than kCfHalo / 2 samples per group: not with this geometry) is served from global
// memory by cf_window_global.  (The first version -- head flags, a device-wide scan for the group numbers, a group start table
// and a per-sample chain of dependent L1 / L2 lookups -- took 4.9 ms for the 1.06e8 samples of a 1 ms cut.)
// Algorithmic HBM bytes: 16 per sample read + 16 per cluster written.  All arithmetic fp32 in the written order (--fmad=false).
#pragma once
#include "common.cuh"
#include "scan.cuh"

namespace tpc {

struct CfDigits { const int32_t* row; const int32_t* pad; const int32_t* time; const float* adc; };
struct CfOut { int64_t max_clusters; float *row, *pad, *time, *charge; int64_t* n_clusters; int32_t* status; };
struct CfStage { float *pad, *time, *charge; int32_t* row; };      // [n] each: cluster j of tile t sits at t * kCfTile + j

constexpr int kCfThreads = 256;
constexpr int kCfItems = 8;
constexpr int kCfTile = kCfThreads * kCfItems;        // 2048 samples per CTA
constexpr int kCfHalo = 352;                          // >= 2 x 173 pads (the widest pad row of the default geometry)
constexpr int kCfWin = kCfTile + 2 * kCfHalo;         // 2752 staged samples
constexpr int kCfChunk = (kCfWin + kCfThreads - 1) / kCfThreads;   // 11 window entries per thread in the running-maximum pass

struct CfSmem {
  int32_t pad[kCfWin];
  float adc[kCfWin];
  uint16_t gs[kCfWin];      // window index of the first sample of the entry's group (a TRUE start iff that entry's flag bit 0 is set)
  uint16_t ge[kCfWin];      // at a group's first entry: window index one past its last sample (kCfWin may mean "goes on")
  uint8_t flag[kCfWin];     // bit 0: first sample of its (sector_row, time bin); bit 1: ... and that group is the time bin right
                            // after the group before it, same sector_row
  uint16_t list[kCfTile];   // window indices of the tile's samples at or above the threshold, in input order
  uint32_t warp_max[kCfThreads / 32];
  uint32_t cnt[2 * (kCfThreads / 32)];
};

// The window of sample i, served from global memory (any group size): linear walks to the neighbouring groups, bounded by
// the group sizes.  Returns the peak decision; the sums in the order of D5.
__device__ __noinline__ bool cf_window_global(const CfDigits d, int64_t n, int64_t i, float& q, float& sp, float& st) {
  const int r = d.row[i], p = d.pad[i], t = d.time[i];
  const float a0 = d.adc[i];
  bool peak = true;
  q = sp = st = 0.0f;
  int64_t gs = i;
  while (gs > 0 && d.row[gs - 1] == r && d.time[gs - 1] == t) --gs;
  int64_t ge = i + 1;
  while (ge < n && d.row[ge] == r && d.time[ge] == t) ++ge;
  for (int dt = -1; dt <= 1; ++dt) {
    int64_t a = 0, b = 0;
    if (dt == 0) { a = max(gs, i - 1); b = min(ge, i + 2); }
    else if (dt < 0) {
      if (gs > 0 && d.row[gs - 1] == r && d.time[gs - 1] == t - 1) {
        b = gs; a = gs;
        while (a > 0 && d.row[a - 1] == r && d.time[a - 1] == t - 1 && d.pad[a - 1] >= p - 1) --a;
      }
    } else if (ge < n && d.row[ge] == r && d.time[ge] == t + 1) {
      a = ge; b = ge;
      while (b < n && d.row[b] == r && d.time[b] == t + 1 && d.pad[b] <= p + 1) ++b;
    }
    for (int64_t e = a; e < b; ++e) {
      const int dp = d.pad[e] - p;
      if (dp < -1 || dp > 1) continue;
      const float x = d.adc[e];
      if (e != i && !(a0 > x || (a0 == x && i < e))) peak = false;
      q = q + x;
      sp = sp + (float)dp * x;
      st = st + (float)dt * x;
    }
  }
  return peak;
}

// One tile per CTA (see the header).  Window entry w holds sample w0 + w, w0 = tile start - kCfHalo; entries outside [0, n)
// are invalid and belong to no group.
__global__ void __launch_bounds__(kCfThreads, 4) k_cf_tile(CfDigits d, int64_t n, float thr, CfStage stage, uint32_t* __restrict__ tile_count) {
  extern __shared__ __align__(16) unsigned char cf_smem_raw[];
  CfSmem& s = *reinterpret_cast<CfSmem*>(cf_smem_raw);
  const int tx = threadIdx.x;
  const unsigned lane = lane_id();
  const int wid = tx >> 5;
  const int64_t t0 = (int64_t)blockIdx.x * kCfTile;
  const int64_t w0 = t0 - kCfHalo;
  const int w_first = (int)max((int64_t)0, -w0);                       // first valid window entry
  const int w_end = (int)min((int64_t)kCfWin, n - w0);                 // one past the last valid one
  const bool open_hi = w0 + kCfWin < n;                                // the input goes on behind the window

  // 1. stage the window (coalesced); the group structure comes from comparing every sample with the one before it
  for (int w = tx; w < kCfWin; w += kCfThreads) {
    const bool in = w >= w_first && w < w_end;
    const int64_t g = w0 + w;
    uint8_t f = 1;                                                     // invalid entries are groups of their own
    if (in) {
      s.pad[w] = d.pad[g]; s.adc[w] = d.adc[g];
      if (g > 0) {
        const int r = d.row[g], t = d.time[g], rb = d.row[g - 1], tb = d.time[g - 1];
        f = (r != rb || t != tb) ? (uint8_t)(1 | ((r == rb && t == tb + 1) ? 2 : 0)) : (uint8_t)0;
      }
    } else {
      s.pad[w] = 0; s.adc[w] = 0.0f;
    }
    s.flag[w] = f;
    s.ge[w] = (uint16_t)kCfWin;
  }
  __syncthreads();

  // 2. group starts: gs[w] = the largest head index <= w (entry 0 counts as one), a block-wide running maximum over
  // contiguous chunks
  {
    const int c0 = tx * kCfChunk;
    uint32_t run = 0;
#pragma unroll
    for (int k = 0; k < kCfChunk; ++k) { const int w = c0 + k; if (w < kCfWin && (s.flag[w] & 1)) run = (uint32_t)w; }
    uint32_t inc = run;                                                // inclusive maximum over the threads of the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o); if ((int)lane >= o) inc = max(inc, v); }
    if (lane == 31) s.warp_max[wid] = inc;
    __syncthreads();
    uint32_t pre = __shfl_up_sync(0xffffffffu, inc, 1);
    if (lane == 0) pre = 0;
    for (int ww = 0; ww < wid; ++ww) pre = max(pre, s.warp_max[ww]);
    run = pre;
#pragma unroll
    for (int k = 0; k < kCfChunk; ++k) {
      const int w = c0 + k;
      if (w < kCfWin) { if (s.flag[w] & 1) run = (uint32_t)w; s.gs[w] = (uint16_t)run; }
    }
  }
  __syncthreads();
  // 3. group ends, stored at the group's first entry; and the ordered list of the tile's samples at or above the threshold
  for (int w = tx + 1; w < kCfWin; w += kCfThreads)
    if (s.flag[w] & 1) s.ge[s.gs[w - 1]] = (uint16_t)w;
  uint32_t n_list = 0;
  for (int k = 0; k < kCfItems; ++k) {
    const int w = kCfHalo + k * kCfThreads + tx;
    const bool above = w < w_end && s.adc[w] >= thr;                   // (w >= w_first always: w >= kCfHalo)
    const unsigned bal = __ballot_sync(0xffffffffu, above);
    uint32_t* cnt = s.cnt + (k & 1) * (kCfThreads / 32);
    if (lane == 0) cnt[wid] = __popc(bal);
    __syncthreads();
    uint32_t pre = 0, tot = 0;
#pragma unroll
    for (int ww = 0; ww < kCfThreads / 32; ++ww) { const uint32_t c = cnt[ww]; if (ww < wid) pre += c; tot += c; }
    if (above) s.list[n_list + pre + __popc(bal & ((1u << lane) - 1u))] = (uint16_t)w;
    n_list += tot;
  }
  __syncthreads();

  // 4. one listed sample per thread and round: decision + sums from shared memory, then the round's peaks are written in
  // order -- position = peaks of the earlier rounds + of the lower warps + of the lower lanes (one barrier per round)
  uint32_t base = 0;
  for (uint32_t j0 = 0; j0 < n_list; j0 += kCfThreads) {
    const uint32_t jj = j0 + (uint32_t)tx;
    float q = 0.0f, sp = 0.0f, st = 0.0f;
    bool peak = false;
    int w = 0;
    if (jj < n_list) {
      w = s.list[jj];
      const float a0 = s.adc[w];
      const int p = s.pad[w];
      const int gsw = s.gs[w], gew = s.ge[gsw];
      // are the groups of the window completely staged?
      bool safe = (s.flag[gsw] & 1) && (gew < kCfWin || !open_hi);
      int pa = 0, pb = 0, na = 0, nb = 0;                              // spans of the time bins t - 1 and t + 1
      if (safe && (s.flag[gsw] & 2)) {                                 // the time bin before exists: is it staged from its first sample on?
        if (gsw == 0) safe = false; else { pa = s.gs[gsw - 1]; pb = gsw; safe = s.flag[pa] & 1; }
      }
      if (safe && gew < w_end && (s.flag[gew] & 2)) { na = gew; nb = s.ge[gew]; safe = nb < kCfWin || !open_hi; }
      peak = true;
      if (!safe) {
        peak = cf_window_global(d, n, w0 + w, q, sp, st);
      } else {
        // the window in the order of D5 (dt outer, dp inner): per time bin the first entry with pad >= p - 1, then three probes
#pragma unroll
        for (int dt = -1; dt <= 1; ++dt) {
          int a, hi;
          if (dt == 0) { a = max(gsw, w - 1); hi = min(gew, w + 2); }
          else {
            a = dt < 0 ? pa : na; hi = dt < 0 ? pb : nb;
            int b = hi;
            while (a < b) { const int m = (a + b) >> 1; if (s.pad[m] < p - 1) a = m + 1; else b = m; }
          }
#pragma unroll
          for (int e3 = 0; e3 < 3; ++e3) {
            const int e = a + e3;
            const int ec = min(e, kCfWin - 1);
            const int dp = s.pad[ec] - p;
            const float x = s.adc[ec];
            const bool use = e < hi && dp >= -1 && dp <= 1;
            if (use && e != w && !(a0 > x || (a0 == x && w < e))) peak = false;
            q = use ? q + x : q;
            sp = use ? sp + (float)dp * x : sp;
            st = use ? st + (float)dt * x : st;
          }
        }
      }
    }
    const unsigned bal = __ballot_sync(0xffffffffu, peak);
    uint32_t* cnt = s.cnt + ((j0 / kCfThreads) & 1) * (kCfThreads / 32);
    if (lane == 0) cnt[wid] = __popc(bal);
    __syncthreads();
    uint32_t pre = 0, tot = 0;
#pragma unroll
    for (int ww = 0; ww < kCfThreads / 32; ++ww) { const uint32_t c = cnt[ww]; if (ww < wid) pre += c; tot += c; }
    if (peak) {
      const int64_t j = t0 + base + pre + __popc(bal & ((1u << lane) - 1u));
      const int64_t g = w0 + w;
      stage.row[j] = d.row[g];
      stage.pad[j] = (float)s.pad[w] + sp / q;
      stage.time[j] = (float)d.time[g] + st / q;
      stage.charge[j] = q;
    }
    base += tot;
  }
  if (tx == 0) tile_count[blockIdx.x] = base;
}

// tile_off = exclusive scan of tile_count, *total behind it.  One CTA per tile copies its staged clusters to their final place.
__global__ void __launch_bounds__(kCfThreads) k_cf_compact(CfStage stage, const uint32_t* __restrict__ tile_count, const uint32_t* __restrict__ tile_off,
                                                           const uint32_t* __restrict__ total, CfOut o) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    *o.n_clusters = (int64_t)*total;
    *o.status = (int64_t)*total > o.max_clusters ? 1 : 0;       // more clusters than capacity: the first max_clusters are written
  }
  const uint32_t cnt = tile_count[blockIdx.x];
  const int64_t src = (int64_t)blockIdx.x * kCfTile, dst = tile_off[blockIdx.x];
  for (uint32_t j = threadIdx.x; j < cnt; j += kCfThreads) {
    if (dst + j >= o.max_clusters) break;
    o.row[dst + j] = (float)stage.row[src + j];
    o.pad[dst + j] = stage.pad[src + j];
    o.time[dst + j] = stage.time[src + j];
    o.charge[dst + j] = stage.charge[src + j];
  }
}

}  // namespace tpc
