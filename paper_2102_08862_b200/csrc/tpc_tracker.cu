// C-ABI boundary and host orchestration of the B200-native TPC time-frame tracker (include/tpc_tracker.h).
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo --fmad=false -shared -Xcompiler -fPIC
// (--fmad=false: the decision arithmetic must round like the definition, BASELINE.json L5.)
#include "../../include/tpc_tracker.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "arena.h"
#include "clusterizer.cuh"
#include "common.cuh"
#include "compress.cuh"
#include "finder.cuh"
#include "follow_rows.cuh"
#include "ingest.cuh"
#include "links.cuh"
#include "merge.cuh"
#include "fullfit.cuh"
#include "scan.cuh"
#include "selector.cuh"
#include "tracklet.cuh"

using namespace tpc;

namespace {

enum Step {
  S_SORT = 0, S_GRID, S_FINDER, S_CLEAN_START, S_COMPACT,
  S_TL_INIT, S_FIT_UP, S_FOLLOW_UP, S_FIT_DOWN, S_FOLLOW_DOWN,      // C5 tracklet constructor: seed + its four phase kernels
  S_CLAIM, S_COUNT, S_SELECT_SCAN, S_EMIT, N_STEPS
};
const char* const kStepNames[N_STEPS] = {
    "ingest_radix_sort", "grid_build", "neighbours_finder", "cleaner_start_hits", "start_hit_compaction",
    "tracklet_init", "tracklet_fit_up", "tracklet_follow_up", "tracklet_fit_down", "tracklet_follow_down", "selector_claim", "selector_count", "selector_scan", "selector_emit"};

struct Ids {   // arena allocation ids
  int stage_in = -1, stage_out = -1;
  int bin_start, sort_keys, tmp_keys, tmp_orig, tmp_yt, sort_hist, yt, orig, hsr, link_up, link_down, link_up_clean, start_flag, cell_count, start_hits,
      scan_a, scan_b, seeds_a, seeds_b, row_hit, tl_meta, tl_rec, tl_cur, claim, owned,
      flag, track_idx, hit_off, track_slot, chunks, gap_list;
};

struct Capacities {
  int64_t max_clusters, max_tracklets, max_tracks, max_track_hits;
  int n_tb, n_pb, grid_w, n_bins, n_link_ctas;
  int n_slices, slice_bins;     // start-hit processing order: time slices of slice_bins grid time bins
  int64_t n_cells, max_chunks;
  int sort_passes, sort_digit_bits, sort_tiles;
};

constexpr int kDefaultGridTimeBins = 8, kDefaultGridPadBins = 8, kDefaultSliceTimeBins = 256;   // measured: 8 x 8 67.5 ms, 4 x 8 68.6, 6 x 8 67.9, 3 x 8 73.3 (configs[3])
#ifndef TPC_FOLLOW_CTAS_PER_SM
#define TPC_FOLLOW_CTAS_PER_SM 64
#endif
#ifndef TPC_FIT_CTAS_PER_SM
#define TPC_FIT_CTAS_PER_SM 64
#endif
// The grid lookups add ABSOLUTE superset margins to their time windows (0.05 / 0.02 time bins, tracklet.cuh / finder.cuh)
// that must exceed the rounding of a predicted fp32 time: half an ulp at 2^19 bins is 0.03, so frames are limited to
// 2^19 time bins (104 ms; the paper's frame is 10 ms = 5e4 bins).
constexpr float kMaxTimeBin = 524288.0f;
constexpr double kGridMarginCm = 0.01;   // superset margin of the pad-bin lookups (fp32 rounding of a difference is << this)

bool valid_geometry(const tpc_geometry_t* g) {
  return g && g->n_sectors >= 1 && g->n_rows >= 3 && g->n_rows <= kRowStride &&
         (int64_t)g->n_sectors * g->n_rows <= 65535 && g->row_pitch_cm > 0 && g->pad_pitch_cm > 0 &&
         g->tan_half_sector > 0 && g->time_bin_cm > 0 && g->max_time_bin >= 0 && std::isfinite(g->max_time_bin) &&
         g->max_time_bin < kMaxTimeBin;
}

bool valid_params(const tpc_params_t* p) {
  return p && p->miss_limit >= 1 && p->min_hits >= 1 && p->seed_min_hits >= 2 && p->sigma_y_cm > 0 &&
         p->sigma_z_cm > 0 && p->sin_phi_max > 0 && p->sin_phi_max < 1 && p->grid_time_bins >= 0 && p->slice_time_bins >= 0 && p->grid_pad_bins >= 0 && p->grid_pad_bins <= 64 &&
         p->max_clusters >= 0 && p->max_clusters < ((int64_t)1 << 31) && p->max_tracklets >= 0 &&
         p->max_tracklets <= ((int64_t)1 << kKeySlotBits) && p->max_tracks >= 0 && p->max_track_hits >= 0 &&
         p->win_const > 0 && p->win_slope >= 0 && p->chi2_cut > 0;
}

bool capacities(const tpc_geometry_t* g, const tpc_params_t* p, int64_t max_clusters, Capacities& c) {
  c.max_clusters = max_clusters > 0 ? max_clusters : p->max_clusters;
  if (c.max_clusters < 1) c.max_clusters = 1;
  if (c.max_clusters >= ((int64_t)1 << 31)) return false;
  c.max_tracklets = p->max_tracklets > 0 ? p->max_tracklets : std::min<int64_t>(c.max_clusters / 10 + 4096, (int64_t)1 << kKeySlotBits);   // a claim word carries the slot in 24 bits
  c.max_tracks = p->max_tracks > 0 ? p->max_tracks : c.max_clusters / 64 + 4096;
  c.max_track_hits = p->max_track_hits > 0 ? p->max_track_hits : c.max_clusters;
  // Pad bins per row: as requested, but a lookup window must never span more than two of them.  Widest windows:
  // the finder's search area A_y and the follower's window after miss_limit missed rows, each with its margin.
  {
    const double pitch = (double)g->row_pitch_cm;
    const double w1 = (double)p->win_slope * pitch + (double)p->win_const;
    const double ay = (double)p->slope_y_max * pitch + w1 + kGridMarginCm;
    const double wf = (double)p->win_slope * pitch * (double)(p->miss_limit + 1) + (double)p->win_const + kGridMarginCm;
    const double narrowest = std::floor(2.0 * (double)g->x0_cm * (double)g->tan_half_sector / (double)g->pad_pitch_cm) * (double)g->pad_pitch_cm;
    int npb = p->grid_pad_bins > 0 ? p->grid_pad_bins : kDefaultGridPadBins;
    while (npb > 1 && 2.0 * std::max(ay, wf) * 1.01 > narrowest / (double)npb) --npb;
    c.n_pb = npb;
  }
  // Time bins per grid bin: as requested; by default kDefaultGridTimeBins, widened by up to a quarter if that makes the sort key
  // (the grid bin index) one radix digit size cheaper -- configs[3] at 8 time bins has 2.76e8 bins = 29 bits = four 8-bit passes,
  // at 9 it has 2.45e8 = 28 bits = four 7-bit passes (ingest 8.7 -> 7.4 ms; the searches see 5 % more candidates, +0.1 ms each).
  auto key_bits = [&](int w) {
    const double nbw = (std::floor((double)g->max_time_bin / (double)w) + 1.0) * (double)c.n_pb * (double)g->n_sectors * (double)g->n_rows;
    int b = 1;
    while (std::ldexp(1.0, b) <= nbw) ++b;                            // the sentinel key n_bins must be representable
    return b;
  };
  auto sort_cost = [&](int w) { const int b = key_bits(w), passes = (b + kRadixMaxBits - 1) / kRadixMaxBits; return passes * 16 + (b + passes - 1) / passes; };
  c.grid_w = p->grid_time_bins > 0 ? p->grid_time_bins : kDefaultGridTimeBins;
  if (p->grid_time_bins <= 0)
    for (int w = kDefaultGridTimeBins + 1; w <= kDefaultGridTimeBins + kDefaultGridTimeBins / 4; ++w)
      if (sort_cost(w) < sort_cost(c.grid_w)) c.grid_w = w;
  const double ntb = std::floor((double)g->max_time_bin / (double)c.grid_w) + 1.0;
  const double nb = ntb * (double)c.n_pb * (double)g->n_sectors * (double)g->n_rows;
  if (nb >= 2147483000.0) return false;
  c.n_tb = (int)ntb;
  c.n_bins = (int)nb;
  c.n_link_ctas = (int)((c.max_clusters + kLinkThreads - 1) / kLinkThreads);
  const int slice_tb = p->slice_time_bins > 0 ? p->slice_time_bins : kDefaultSliceTimeBins;
  c.slice_bins = std::max(1, slice_tb / c.grid_w);
  c.n_slices = (c.n_tb + c.slice_bins - 1) / c.slice_bins;
  c.n_cells = (int64_t)g->n_sectors * g->n_rows * c.n_slices;
  if (c.n_cells >= 2147483000) return false;
  c.max_chunks = c.max_tracklets / kFrChunk + (int64_t)g->n_sectors * c.n_slices + 2;      // follow_rows.cuh: chunks never straddle a (sector, slice) group
  int bits = 1;
  while (((int64_t)1 << bits) <= (int64_t)c.n_bins) ++bits;          // the sentinel key n_bins must be representable
  c.sort_passes = (bits + kRadixMaxBits - 1) / kRadixMaxBits;
  c.sort_digit_bits = (bits + c.sort_passes - 1) / c.sort_passes;
  c.sort_tiles = (int)((c.max_clusters + kRadixTile - 1) / kRadixTile);
  return true;
}

void build_plan(const tpc_params_t* p, const Capacities& c, ArenaPlan& plan, Ids& id) {
  const size_t N = (size_t)c.max_clusters, T = (size_t)c.max_tracklets, B = (size_t)c.n_bins + 1;
  if (p->host_staging) {
    id.stage_in = plan.add("host_staging_in(row,pad,time)", 3 * 4 * N, S_SORT, S_SORT);
    const size_t K = (size_t)c.max_tracks;
    id.stage_out = plan.add("host_staging_out(tracks)", 256 + K * (5 * 4 + 8 + 7 * 4 + 9 * 4) + 4 * (size_t)c.max_track_hits + 64,
                            S_EMIT, S_EMIT);
  }
  const size_t hist_len = (size_t)kRadixBuckets * (size_t)c.sort_tiles + 1;
  const size_t scan_len = std::max(std::max(scan_tiles(hist_len), scan_tiles((size_t)c.n_cells + 1)), scan_tiles(T)) + 2;
  id.scan_a = plan.add("scan_tile_sums_a", 4 * scan_len, S_SORT, S_EMIT);
  id.scan_b = plan.add("scan_tile_sums_b", 4 * scan_len, S_SORT, S_EMIT);
  id.bin_start = plan.add("grid_bin_start", 4 * B, S_GRID, S_COUNT);        // its last entry (= number of valid hits) is read up to the count step
  id.sort_keys = plan.add("sort_keys", 4 * N, S_SORT, S_GRID);
  // long runs of empty bins, cut into segments: <= one per kGridGapSegment bins + one per run longer than kGridGapInline
  id.gap_list = plan.add("grid_gap_segments(uint4)", 16 * ((size_t)c.n_bins / kGridGapSegment + std::min<size_t>(N + 1, (size_t)c.n_bins / kGridGapInline) + 2), S_GRID, S_GRID);
  id.tmp_keys = plan.add("sort_tmp_keys", 4 * N, S_SORT, S_SORT);
  id.tmp_orig = plan.add("sort_tmp_orig", 4 * N, S_SORT, S_SORT);
  id.tmp_yt = plan.add("sort_tmp_y_time", 8 * N, S_SORT, S_SORT);
  id.sort_hist = plan.add("sort_tile_histograms", 4 * hist_len, S_SORT, S_SORT);
  id.yt = plan.add("hits_y_time(float2)", 8 * N, S_SORT, S_EMIT);      // the emit kernel copies the track hits' (y, time) on request
  id.orig = plan.add("hits_orig_index", 4 * N, S_SORT, S_EMIT);
  id.hsr = plan.add("hits_sector_row(u16)", 2 * N, S_GRID, S_EMIT);
  id.link_up = plan.add("link_up_raw", 4 * N, S_FINDER, S_CLEAN_START);
  id.link_down = plan.add("link_down_raw", 4 * N, S_FINDER, S_CLEAN_START);
  id.link_up_clean = plan.add("link_up_clean", 4 * N, S_CLEAN_START, S_TL_INIT);
  id.start_flag = plan.add("start_flag(u8)", N, S_CLEAN_START, S_COMPACT);
  id.cell_count = plan.add("start_cell_count", 4 * ((size_t)c.n_cells + 2), S_COMPACT, S_COMPACT);
  id.start_hits = plan.add("start_hits", 4 * T, S_COMPACT, S_EMIT);
  id.chunks = plan.add("follower_chunks(uint2)", 8 * (size_t)c.max_chunks, S_COMPACT, S_FOLLOW_DOWN);
  id.seeds_a = plan.add("tracklet_seeds_a(int4)", 16 * T, S_TL_INIT, S_FOLLOW_DOWN);
  id.seeds_b = plan.add("tracklet_seeds_b(float4)", 16 * T, S_TL_INIT, S_FOLLOW_DOWN);
  id.row_hit = plan.add("tracklet_row_hit", 4 * (size_t)kRowStride * T, S_TL_INIT, S_EMIT);
  id.tl_meta = plan.add("tracklet_meta(int4)", 16 * T, S_FIT_UP, S_EMIT);
  id.tl_rec = plan.add("tracklet_record(4 x float4)", 64 * T, S_FIT_UP, S_EMIT);
  id.tl_cur = plan.add("tracklet_handover(2 x float4)", 32 * T, S_FOLLOW_UP, S_FIT_DOWN);
  id.claim = plan.add("selector_claim(u64)", 8 * N, S_CLAIM, S_EMIT);      // emit re-reads the claims of the tracks' hits
  id.owned = plan.add("selector_owned", 4 * T, S_COUNT, S_EMIT);
  id.flag = plan.add("selector_flag", 4 * T, S_COUNT, S_EMIT);
  id.track_idx = plan.add("selector_track_idx", 4 * T, S_SELECT_SCAN, S_EMIT);
  id.hit_off = plan.add("selector_hit_off", 4 * T, S_SELECT_SCAN, S_EMIT);
  id.track_slot = plan.add("selector_track_slot", 4 * T, S_EMIT, S_EMIT);
  plan.plan();
}

}  // namespace

// C7 scratch (merge.cuh), carved from the start of the arena: the tracking scratch is dead by then.
namespace {
struct MergeLayout { size_t cell_start, cell_cursor, scan, cell_of, cand_idx, cand_a, cand_b, out_key, out_b, in_key, out_t, total; int n_tcell; size_t n_cells; };
MergeLayout merge_layout(const tpc_geometry_t& g, int64_t max_tracks) {
  MergeLayout L{};
  L.n_tcell = (int)std::floor((double)g.max_time_bin / (double)kMergeCellTimeBins) + 2;
  L.n_cells = (size_t)g.n_sectors * (size_t)g.n_rows * (size_t)L.n_tcell;
  const size_t K = (size_t)std::max<int64_t>(max_tracks, 1);
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
  L.cell_start = take(4 * (L.n_cells + 1));
  L.cell_cursor = take(4 * L.n_cells);
  L.scan = take(4 * (scan_tiles(L.n_cells + 1) + 1));
  L.cell_of = take(4 * K);
  L.cand_idx = take(4 * K);
  L.cand_a = take(16 * K);
  L.cand_b = take(8 * K);
  L.out_key = take(8 * K);
  L.out_b = take(4 * K);
  L.in_key = take(8 * K);
  L.out_t = take(4 * K);
  L.total = off;
  return L;
}
}  // namespace

struct tpc_tracker {
  tpc_geometry_t geom;
  tpc_params_t params;
  Capacities cap;
  ArenaPlan plan;
  Ids id;
  Consts consts;
  void* tables = nullptr;          // device: xr | cr | npads
  int32_t* counters = nullptr;     // device: the 256-byte counter block of the last tpc_track_timeframe call (inside `tables`, NOT in
                                   // the arena: tpc_merge_tracks / tpc_refit_chains reuse the arena from offset 0)
  cudaEvent_t ev[N_STEPS + 1] = {};
  bool profile = false, have_times = false;
  int64_t last_launches = 0, last_merge_launches = 0;
  int ctas_refit = 148 * 8, ctas_fullfit = 148 * 4;
  int ctas_fit_up = 148, ctas_follow_up = 148, ctas_fit_down = 148, ctas_follow_down = 148;   // persistent grids: SMs x resident CTAs per SM
  int ctas_rows_up = 148, ctas_rows_down = 148;
  bool follow_rows = false;        // row-synchronous follower (follow_rows.cuh) instead of the per-lane one
};

// Exhaustive check of sqrt_rn_normal / rcp_rn_normal (tracklet.cuh) against sqrtf() / (1.0f / x) over every fp32 bit
// pattern of their stated ranges; counts the mismatching patterns (expected: 0, 0).
__global__ void __launch_bounds__(256) k_selftest_fast_math(unsigned long long* __restrict__ mismatches) {
  unsigned long long bad_sqrt = 0, bad_rcp = 0;
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  for (uint64_t b = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; b < (1ull << 32); b += stride) {
    const uint32_t bits = (uint32_t)b;
    const float x = __uint_as_float(bits);
    if (bits >= 0x0d000000u && bits <= 0x7f7fffffu)                       // [2^-101, FLT_MAX]
      if (__float_as_uint(sqrt_rn_normal(x)) != __float_as_uint(sqrtf(x))) ++bad_sqrt;
    const uint32_t e = (bits >> 23) & 0xffu;
    if (e >= 1u && e <= 252u)                                             // |x| in [2^-126, 2^126)
      if (__float_as_uint(rcp_rn_normal(x)) != __float_as_uint(1.0f / x)) ++bad_rcp;
  }
  bad_sqrt = __reduce_add_sync(0xffffffffu, (unsigned)bad_sqrt);
  bad_rcp = __reduce_add_sync(0xffffffffu, (unsigned)bad_rcp);
  if (lane_id() == 0) { if (bad_sqrt) atomicAdd(mismatches, bad_sqrt); if (bad_rcp) atomicAdd(mismatches + 1, bad_rcp); }
}

// fp32 issue-rate micro-benchmarks (tpc_selftest_alu_peak): 8 independent chains per thread, alternating multiply and add,
// compiled with --fmad=false like the rest of the file, so nothing contracts into FMA.
constexpr int kAluIters = 2048, kAluChains = 8;
__global__ void __launch_bounds__(256) k_alu_peak_scalar(float* __restrict__ sink, float a, float b) {
  float v[kAluChains];
#pragma unroll
  for (int k = 0; k < kAluChains; ++k) v[k] = (float)(threadIdx.x + k) * 1.0e-3f;
  for (int i = 0; i < kAluIters; ++i) {
#pragma unroll
    for (int k = 0; k < kAluChains; ++k) v[k] = v[k] * a;
#pragma unroll
    for (int k = 0; k < kAluChains; ++k) v[k] = v[k] + b;
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < kAluChains; ++k) s += v[k];
  if (s == 123.456f) sink[blockIdx.x] = s;             // never true: keeps the chains alive
}
// Packed form: every multiply is fma.rn.f32x2(a, b, -0) and every add fma.rn.f32x2(a, 1, c) -- exactly RN(a*b) and RN(a+c)
// in both halves (IEEE), written as explicit FMAs because ptxas contracts a mul.rn.f32x2 feeding an add.rn.f32x2 into one
// FFMA2 even under --fmad=false (seen in the SASS), and an explicit fma is never re-fused.
__global__ void __launch_bounds__(256) k_alu_peak_packed(float* __restrict__ sink, float a, float b) {
  unsigned long long v[kAluChains], pa, pb, one, nz;
  asm("mov.b64 %0, {%1, %1};" : "=l"(pa) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(pb) : "f"(b));
  asm("mov.b64 %0, {%1, %1};" : "=l"(one) : "f"(1.0f));
  asm("mov.b64 %0, {%1, %1};" : "=l"(nz) : "f"(-0.0f));
#pragma unroll
  for (int k = 0; k < kAluChains; ++k) { const float x = (float)(threadIdx.x + k) * 1.0e-3f; asm("mov.b64 %0, {%1, %1};" : "=l"(v[k]) : "f"(x)); }
  for (int i = 0; i < kAluIters; ++i) {
#pragma unroll
    for (int k = 0; k < kAluChains; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v[k]) : "l"(pa), "l"(nz));
#pragma unroll
    for (int k = 0; k < kAluChains; ++k) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v[k]) : "l"(one), "l"(pb));
  }
  float s = 0.0f;
#pragma unroll
  for (int k = 0; k < kAluChains; ++k) { float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v[k])); s += lo + hi; }
  if (s == 123.456f) sink[blockIdx.x] = s;
}

extern "C" {

const char* tpc_strerror(int code) {
  switch (code) {
    case TPC_OK: return "ok";
    case TPC_EINVAL: return "invalid argument";
    case TPC_ENOMEM: return "scratch arena missing or too small";
    case TPC_ECUDA: return "CUDA error (no device, launch or runtime failure)";
    default: return "unknown status";
  }
}

const char* tpc_tracker_step_name(int32_t step) { return step >= 0 && step < N_STEPS ? kStepNames[step] : nullptr; }

size_t tpc_tracker_arena_bytes(const tpc_geometry_t* g, const tpc_params_t* p, int64_t max_clusters) {
  if (!valid_geometry(g) || !valid_params(p)) return 0;
  Capacities c;
  if (!capacities(g, p, max_clusters, c)) return 0;
  ArenaPlan plan;
  Ids id;
  build_plan(p, c, plan, id);
  // the arena also serves tpc_merge_tracks (C7) for the default track capacity
  return std::max(plan.peak_bytes(), merge_layout(*g, c.max_tracks).total);
}

int tpc_tracker_create(const tpc_geometry_t* g, const tpc_params_t* p, tpc_tracker_t** out) {
  if (!out) return TPC_EINVAL;
  *out = nullptr;
  if (!valid_geometry(g) || !valid_params(p)) return TPC_EINVAL;
  tpc_tracker* t = new (std::nothrow) tpc_tracker();
  if (!t) return TPC_ENOMEM;
  t->geom = *g;
  t->params = *p;
  if (!capacities(g, p, 0, t->cap)) { delete t; return TPC_EINVAL; }
  build_plan(p, t->cap, t->plan, t->id);
  if (!p->arena || p->arena_bytes < t->plan.peak_bytes() || (reinterpret_cast<uintptr_t>(p->arena) & 255)) { delete t; return TPC_ENOMEM; }

  // per-row tables in double, rounded once
  const int nr = g->n_rows;
  std::vector<float> xr(nr), cr(nr), yoff(nr), pscale(nr);
  std::vector<int> npads(nr);
  const double pitch = (double)g->row_pitch_cm;
  for (int r = 0; r < nr; ++r) {
    const double x = (double)g->x0_cm + pitch * (double)r;
    xr[r] = (float)x;
    npads[r] = (int)std::floor(2.0 * x * (double)g->tan_half_sector / (double)g->pad_pitch_cm);
    if (npads[r] < 1) { delete t; return TPC_EINVAL; }
    cr[r] = (float)(0.5 * (double)(npads[r] - 1));
    const double width = (double)npads[r] * (double)g->pad_pitch_cm;       // y spans [-width/2, +width/2)
    yoff[r] = (float)(0.5 * width);
    pscale[r] = (float)((double)t->cap.n_pb / width);
  }
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) { cudaGetLastError(); delete t; return TPC_ECUDA; }
  const size_t rowtab_off = ((size_t)nr * 20 + 15) / 16 * 16;      // float4 (npads - 0.5, cr, yoff, pscale) per row, for the ingest key
  const size_t counters_off = (rowtab_off + (size_t)nr * 16 + 255) / 256 * 256;
  const size_t tab_bytes = counters_off + 256;
  std::vector<float> rowtab((size_t)nr * 4);
  for (int r = 0; r < nr; ++r) { rowtab[4 * r] = (float)npads[r] - 0.5f; rowtab[4 * r + 1] = cr[r]; rowtab[4 * r + 2] = yoff[r]; rowtab[4 * r + 3] = pscale[r]; }
  if (cudaMalloc(&t->tables, tab_bytes) != cudaSuccess) { cudaGetLastError(); delete t; return TPC_ECUDA; }
  char* tb = static_cast<char*>(t->tables);
  if (cudaMemcpy(tb, xr.data(), (size_t)nr * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(tb + (size_t)nr * 4, cr.data(), (size_t)nr * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(tb + (size_t)nr * 8, npads.data(), (size_t)nr * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(tb + (size_t)nr * 12, yoff.data(), (size_t)nr * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(tb + (size_t)nr * 16, pscale.data(), (size_t)nr * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(tb + rowtab_off, rowtab.data(), (size_t)nr * 16, cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaGetLastError(); cudaFree(t->tables); delete t; return TPC_ECUDA;
  }

  t->counters = reinterpret_cast<int32_t*>(tb + counters_off);
  if (cudaMemset(t->counters, 0, 256) != cudaSuccess) { cudaGetLastError(); cudaFree(t->tables); delete t; return TPC_ECUDA; }
  Consts& c = t->consts;
  const int w = t->cap.grid_w;
  c.n_rows = nr; c.n_sr = g->n_sectors * nr; c.n_tb = t->cap.n_tb; c.n_pb = t->cap.n_pb; c.n_bins = t->cap.n_bins;
  c.max_time = g->max_time_bin; c.inv_bin_w = (float)(1.0 / (double)w); c.inv_n_rows = (float)(1.0 / (double)nr);
  c.Z = g->time_bin_cm; c.inv_Z = (float)(1.0 / (double)g->time_bin_cm); c.P = g->pad_pitch_cm;
  const double w1 = (double)p->win_slope * pitch + (double)p->win_const;
  c.W1 = (float)w1;
  c.Ay = (float)((double)p->slope_y_max * pitch + w1);
  c.Az = (float)((double)p->slope_z_max * pitch + w1);
  const double sy2 = (double)p->sigma_y_cm * (double)p->sigma_y_cm, sz2 = (double)p->sigma_z_cm * (double)p->sigma_z_cm;
  c.wy = (float)(1.0 / (6.0 * sy2)); c.wz = (float)(1.0 / (6.0 * sz2));
  c.ry = (float)sy2; c.rz = (float)sz2;
  c.chi2_cut = p->chi2_cut;
  c.finder_tw = (float)((double)c.Az / (double)g->time_bin_cm + 0.02);
  c.finder_yw = (float)((double)c.Ay + kGridMarginCm);
  c.cB = p->inv_R_per_qpt; c.sin_phi_max = p->sin_phi_max; c.win_slope = p->win_slope; c.win_const = p->win_const;
  c.c0_y2 = p->c0_y2; c.c0_s2 = p->c0_s2; c.c0_k2 = p->c0_k2; c.c0_z2 = p->c0_z2; c.c0_t2 = p->c0_t2;
  c.miss_limit = p->miss_limit; c.min_hits = p->min_hits; c.seed_min_hits = p->seed_min_hits;
  c.xr = reinterpret_cast<const float*>(tb);
  c.cr = reinterpret_cast<const float*>(tb + (size_t)nr * 4);
  c.npads = reinterpret_cast<const int*>(tb + (size_t)nr * 8);
  c.yoff = reinterpret_cast<const float*>(tb + (size_t)nr * 12);
  c.pscale = reinterpret_cast<const float*>(tb + (size_t)nr * 16);
  c.rowtab = reinterpret_cast<const float4*>(tb + rowtab_off);

  t->profile = p->profile != 0;
  if (cudaFuncSetAttribute(k_radix_scatter<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRadixScatterSmem) != cudaSuccess ||
      cudaFuncSetAttribute(k_radix_scatter<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRadixScatterSmem) != cudaSuccess) {
    cudaGetLastError(); tpc_tracker_destroy(t); return TPC_ECUDA;
  }
  {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    auto resident = [&](auto kernel, int cap) {
      int per_sm = 1;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kTrackletThreads, 0) != cudaSuccess || per_sm < 1) {
        cudaGetLastError(); per_sm = 1;
      }
      return sms * std::min(per_sm, cap);
    };
    t->ctas_fit_up = resident(k_tracklet_fit<false>, TPC_FIT_CTAS_PER_SM);
    t->ctas_follow_up = resident(k_tracklet_follow<false>, TPC_FOLLOW_CTAS_PER_SM);
    t->ctas_fit_down = resident(k_tracklet_fit<true>, TPC_FIT_CTAS_PER_SM);
    t->ctas_follow_down = resident(k_tracklet_follow<true>, TPC_FOLLOW_CTAS_PER_SM);
    t->ctas_refit = resident(k_refit_chains, 64);
    t->ctas_fullfit = resident(k_refit_full, 64);
    t->follow_rows = p->follower == 1 && p->miss_limit <= 255;      // the packed per-tracklet counters are 8 bits wide
    if (cudaFuncSetAttribute(k_cf_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(CfSmem)) != cudaSuccess) {
      cudaGetLastError(); tpc_tracker_destroy(t); return TPC_ECUDA;
    }
    if (cudaFuncSetAttribute(k_follow_rows<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FrSmem)) != cudaSuccess ||
        cudaFuncSetAttribute(k_follow_rows<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FrSmem)) != cudaSuccess) {
      cudaGetLastError(); tpc_tracker_destroy(t); return TPC_ECUDA;
    }
    auto resident_rows = [&](auto kernel) {
      int per_sm = 1;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kFrThreads, sizeof(FrSmem)) != cudaSuccess || per_sm < 1) {
        cudaGetLastError(); per_sm = 1;
      }
      return sms * per_sm;
    };
    t->ctas_rows_up = resident_rows(k_follow_rows<false>);
    t->ctas_rows_down = resident_rows(k_follow_rows<true>);
  }
  for (int i = 0; i <= N_STEPS; ++i)
    if (cudaEventCreate(&t->ev[i]) != cudaSuccess) { cudaGetLastError(); tpc_tracker_destroy(t); return TPC_ECUDA; }
  *out = t;
  return TPC_OK;
}


// ---- C7: sector-boundary merging of the tracks of one tpc_track_timeframe call (merge.cuh) ----

size_t tpc_merge_scratch_bytes(const tpc_tracker_t* t, int64_t max_tracks) {
  if (!t || max_tracks < 0 || max_tracks >= ((int64_t)1 << 31)) return 0;
  return merge_layout(t->geom, max_tracks).total;
}

int tpc_merge_tracks(tpc_tracker_t* t, const tpc_merge_params_t* mp, const tpc_tracks_t* tr, void* cuda_stream, tpc_merged_t* out) {
  if (!t || !mp || !tr || !out) return TPC_EINVAL;
  if (!(mp->cut_y_cm > 0 && mp->cut_z_cm > 0 && mp->cut_sin_phi > 0 && mp->cut_q_pt > 0 && mp->max_row_gap >= 0 && mp->max_row_overlap >= 0)) return TPC_EINVAL;
  if (tr->max_tracks < 0 || !tr->n_tracks || !out->next || !out->prev || !out->root || !out->n_links) return TPC_EINVAL;
  if (tr->max_tracks > 0 && (!tr->seed_hit || !tr->sector || !tr->first_row || !tr->last_row || !tr->x || !tr->y || !tr->z_rel ||
                             !tr->time_ref || !tr->sin_phi || !tr->dzds || !tr->q_pt)) return TPC_EINVAL;
  const MergeLayout L = merge_layout(t->geom, tr->max_tracks);
  if (!t->params.arena || L.total > t->params.arena_bytes) return TPC_ENOMEM;
  if (L.n_cells + 1 >= 2147483000ull) return TPC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* A = static_cast<char*>(t->params.arena);
  const int K = tr->max_tracks;
  MergeConsts c{};
  c.n_sectors = t->geom.n_sectors; c.n_rows = t->geom.n_rows; c.n_tcell = L.n_tcell;
  c.gap = mp->max_row_gap; c.overlap = mp->max_row_overlap; c.max_tracks = K;
  c.x0 = t->geom.x0_cm; c.pitch = t->geom.row_pitch_cm;
  {   // cos / sin of the sector angle from tan of its half, in double, rounded once (no libm: the oracle derives them the same way)
    const double T = (double)t->geom.tan_half_sector;
    c.Cd = (float)((1.0 - T * T) / (1.0 + T * T));
    c.Sd = (float)(2.0 * T / (1.0 + T * T));
  }
  c.Z = t->consts.Z; c.inv_Z = t->consts.inv_Z; c.cB = t->consts.cB; c.sin_phi_max = t->consts.sin_phi_max;
  c.cut_y = mp->cut_y_cm; c.cut_z = mp->cut_z_cm; c.cut_s = mp->cut_sin_phi; c.cut_k = mp->cut_q_pt;
  c.wy = (float)(1.0 / ((double)mp->cut_y_cm * (double)mp->cut_y_cm));
  c.wz = (float)(1.0 / ((double)mp->cut_z_cm * (double)mp->cut_z_cm));
  c.ws = (float)(1.0 / ((double)mp->cut_sin_phi * (double)mp->cut_sin_phi));
  c.wk = (float)(1.0 / ((double)mp->cut_q_pt * (double)mp->cut_q_pt));
  c.inv_cell = 1.0f / (float)kMergeCellTimeBins;
  c.t_window = (float)((double)mp->cut_z_cm / (double)t->geom.time_bin_cm + 0.5);
  c.xr = t->consts.xr;
  MergeTracks T{tr->n_tracks, tr->seed_hit, tr->sector, tr->first_row, tr->last_row, tr->x, tr->y, tr->z_rel, tr->time_ref, tr->sin_phi, tr->dzds, tr->q_pt};
  MergeScratch S{reinterpret_cast<uint32_t*>(A + L.cell_start), reinterpret_cast<uint32_t*>(A + L.cell_cursor),
                 reinterpret_cast<uint32_t*>(A + L.cell_of), reinterpret_cast<uint32_t*>(A + L.cand_idx),
                 reinterpret_cast<float4*>(A + L.cand_a), reinterpret_cast<float2*>(A + L.cand_b),
                 reinterpret_cast<unsigned long long*>(A + L.out_key), reinterpret_cast<int32_t*>(A + L.out_b),
                 reinterpret_cast<unsigned long long*>(A + L.in_key)};
  int64_t launches = 0;
  cudaMemsetAsync(out->n_links, 0, 4, st);
  if (K > 0) {
    cudaMemsetAsync(out->next, 0xFF, 4 * (size_t)K, st);
    cudaMemsetAsync(out->prev, 0xFF, 4 * (size_t)K, st);
    cudaMemsetAsync(out->root, 0xFF, 4 * (size_t)K, st);
    cudaMemsetAsync(S.cell_start, 0, 4 * (L.n_cells + 1), st);
    cudaMemsetAsync(S.cell_cursor, 0, 4 * L.n_cells, st);
    cudaMemsetAsync(S.in_key, 0xFF, 8 * (size_t)K, st);
    const int g256 = (K + 255) / 256;
    k_merge_cell_count<<<g256, 256, 0, st>>>(T, S, c); ++launches;
    launches += exclusive_scan_u32(S.cell_start, S.cell_start, L.n_cells + 1, reinterpret_cast<uint32_t*>(A + L.scan), st);
    k_merge_cell_fill<<<g256, 256, 0, st>>>(T, S, c); ++launches;
    k_merge_match<<<(K + kMergeThreads - 1) / kMergeThreads, kMergeThreads, 0, st>>>(T, S, c); ++launches;
    k_merge_link<<<g256, 256, 0, st>>>(T, S, out->next, out->prev, out->n_links, c); ++launches;
    k_merge_root<<<g256, 256, 0, st>>>(T, out->prev, out->root, c); ++launches;
  }
  t->last_merge_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C0: cluster finder in front of the path (clusterizer.cuh) ----
namespace {
struct CfLayout { size_t st_row, st_pad, st_time, st_charge, tile_count, tile_off, scan_tiles, total; size_t n_tiles; };
CfLayout cf_layout(int64_t n) {
  CfLayout L{};
  const size_t N = (size_t)std::max<int64_t>(n, 1);
  L.n_tiles = (N + kCfTile - 1) / kCfTile;
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
  L.st_row = take(4 * N); L.st_pad = take(4 * N); L.st_time = take(4 * N); L.st_charge = take(4 * N);
  L.tile_count = take(4 * L.n_tiles); L.tile_off = take(4 * L.n_tiles); L.scan_tiles = take(4 * (scan_tiles(L.n_tiles) + 2));
  L.total = off;
  return L;
}
}  // namespace

size_t tpc_cluster_finder_scratch_bytes(int64_t n_digits) {
  if (n_digits < 0 || n_digits >= ((int64_t)1 << 32) - 4096) return 0;
  return cf_layout(n_digits).total;
}

int tpc_find_clusters(tpc_tracker_t* t, const tpc_cluster_params_t* cp, const tpc_digits_t* dg, int64_t n, void* cuda_stream, tpc_clusters_out_t* o) {
  if (!t || !cp || !dg || !o || n < 0 || n >= ((int64_t)1 << 32) - 4096) return TPC_EINVAL;
  if (!(cp->peak_threshold > 0) || !o->n_clusters || !o->status || o->max_clusters < 0) return TPC_EINVAL;
  if (n > 0 && (!dg->row || !dg->pad || !dg->time || !dg->adc)) return TPC_EINVAL;
  if (o->max_clusters > 0 && (!o->row || !o->pad || !o->time || !o->charge)) return TPC_EINVAL;
  const CfLayout L = cf_layout(n);
  if (!t->params.arena || L.total > t->params.arena_bytes) return TPC_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* A = static_cast<char*>(t->params.arena);
  const CfStage stage{reinterpret_cast<float*>(A + L.st_pad), reinterpret_cast<float*>(A + L.st_time), reinterpret_cast<float*>(A + L.st_charge),
                      reinterpret_cast<int32_t*>(A + L.st_row)};
  uint32_t* tile_count = reinterpret_cast<uint32_t*>(A + L.tile_count);
  uint32_t* tile_off = reinterpret_cast<uint32_t*>(A + L.tile_off);
  uint32_t* scan_scratch = reinterpret_cast<uint32_t*>(A + L.scan_tiles);
  int64_t launches = 0;
  if (n == 0) {
    cudaMemsetAsync(o->n_clusters, 0, 8, st);
    cudaMemsetAsync(o->status, 0, 4, st);
  } else {
    const CfDigits d{dg->row, dg->pad, dg->time, dg->adc};
    const CfOut out{o->max_clusters, o->row, o->pad, o->time, o->charge, o->n_clusters, o->status};
    const int n_tiles = (int)L.n_tiles;
    k_cf_tile<<<n_tiles, kCfThreads, sizeof(CfSmem), st>>>(d, n, cp->peak_threshold, stage, tile_count); ++launches;
    launches += exclusive_scan_u32(tile_count, tile_off, (size_t)n_tiles, scan_scratch, st);       // scan_scratch[tiles] = number of clusters
    k_cf_compact<<<n_tiles, kCfThreads, 0, st>>>(stage, tile_count, tile_off, scan_scratch + scan_tiles((size_t)n_tiles), out); ++launches;
  }
  t->last_merge_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C0 without any allocation: the same two kernels with their scratch in a file-scope device array ----
// For callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it) and so cannot
// create a tracker handle with an arena.  The scratch (staged clusters + per-tile counts, 16 B per sample) lives in the
// library image: every GPU that loads the library holds kCfStaticBytes (16.1 MiB) until the process exits.
namespace {
constexpr int64_t kCfStaticMaxDigits = (int64_t)1 << 20;                       // 1 048 576 samples per call
constexpr size_t kCfStaticTiles = (size_t)(kCfStaticMaxDigits / kCfTile);      // 512
constexpr size_t kCfStaticStage = 4 * (size_t)kCfStaticMaxDigits;              // bytes of one staged array
constexpr size_t kCfStaticCounts = 4 * 4 * kCfStaticTiles;                     // tile_count | tile_off | scan scratch (2 + spare)
constexpr size_t kCfStaticBytes = 4 * kCfStaticStage + kCfStaticCounts;
constexpr int kCfStaticMaxDevices = 64;
}  // namespace
static_assert(sizeof(CfSmem) <= 48 * 1024, "k_cf_tile must launch without an opt-in to large dynamic shared memory");
static __device__ __align__(256) unsigned char g_cf_static_scratch[kCfStaticBytes];
namespace {
// In host code g_cf_static_scratch is only a stand-in for the symbol, not a device address: its address on a device comes
// from cudaGetSymbolAddress with that device current, looked up once per device.
std::mutex g_cf_static_mu;
unsigned char* g_cf_static_ptr[kCfStaticMaxDevices] = {};

int cf_static_scratch(unsigned char** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kCfStaticMaxDevices) { cudaGetLastError(); return TPC_ECUDA; }
  std::lock_guard<std::mutex> lock(g_cf_static_mu);
  if (!g_cf_static_ptr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_cf_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return TPC_ECUDA; }
    g_cf_static_ptr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_cf_static_ptr[dev];
  return TPC_OK;
}
}  // namespace

int64_t tpc_find_clusters_static_max_digits(void) { return kCfStaticMaxDigits; }

int tpc_find_clusters_static_setup(void) {
  unsigned char* p = nullptr;
  return cf_static_scratch(&p);
}

int tpc_find_clusters_static(const tpc_cluster_params_t* cp, const tpc_digits_t* dg, int64_t n, void* cuda_stream, tpc_clusters_out_t* o) {
  if (!cp || !dg || !o || n < 0) return TPC_EINVAL;
  if (n > kCfStaticMaxDigits) return TPC_ENOMEM;                               // beyond the built-in scratch: use tpc_find_clusters with an arena
  if (!(cp->peak_threshold > 0) || !o->n_clusters || !o->status || o->max_clusters < 0) return TPC_EINVAL;
  if (n > 0 && (!dg->row || !dg->pad || !dg->time || !dg->adc)) return TPC_EINVAL;
  if (o->max_clusters > 0 && (!o->row || !o->pad || !o->time || !o->charge)) return TPC_EINVAL;
  unsigned char* A = nullptr;
  const int rc = cf_static_scratch(&A);
  if (rc != TPC_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (n == 0) {
    cudaMemsetAsync(o->n_clusters, 0, 8, st);
    cudaMemsetAsync(o->status, 0, 4, st);
  } else {
    const CfStage stage{reinterpret_cast<float*>(A + kCfStaticStage), reinterpret_cast<float*>(A + 2 * kCfStaticStage),
                        reinterpret_cast<float*>(A + 3 * kCfStaticStage), reinterpret_cast<int32_t*>(A)};
    uint32_t* tile_count = reinterpret_cast<uint32_t*>(A + 4 * kCfStaticStage);
    uint32_t* tile_off = tile_count + kCfStaticTiles;
    uint32_t* scan_scratch = tile_off + kCfStaticTiles;
    const CfDigits d{dg->row, dg->pad, dg->time, dg->adc};
    const CfOut out{o->max_clusters, o->row, o->pad, o->time, o->charge, o->n_clusters, o->status};
    const int n_tiles = (int)((n + kCfTile - 1) / kCfTile);
    // the array keeps the last call's contents: the counts start at zero (the staged clusters are written before they are read)
    cudaMemsetAsync(tile_count, 0, kCfStaticCounts, st);
    k_cf_tile<<<n_tiles, kCfThreads, sizeof(CfSmem), st>>>(d, n, cp->peak_threshold, stage, tile_count);
    exclusive_scan_u32(tile_count, tile_off, (size_t)n_tiles, scan_scratch, st);       // scan_scratch[1] = number of clusters (one scan tile)
    k_cf_compact<<<n_tiles, kCfThreads, 0, st>>>(stage, tile_count, tile_off, scan_scratch + scan_tiles((size_t)n_tiles), out);
  }
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C10: merging across the central electrode (merge.cuh) ----
int tpc_merge_central_electrode(tpc_tracker_t* t, const tpc_ce_params_t* mp, const tpc_tracks_t* tr, void* cuda_stream, tpc_ce_merged_t* out) {
  if (!t || !mp || !tr || !out) return TPC_EINVAL;
  if (!(mp->cut_y_cm > 0 && mp->cut_z_cm > 0 && mp->cut_sin_phi > 0 && mp->cut_q_pt > 0 && mp->cut_dzds > 0 && mp->max_row_gap >= 0 &&
        mp->max_row_overlap >= 0)) return TPC_EINVAL;
  if (tr->max_tracks < 0 || !tr->n_tracks || !out->next || !out->prev || !out->t_ce || !out->n_links) return TPC_EINVAL;
  if (tr->max_tracks > 0 && (!tr->seed_hit || !tr->sector || !tr->first_row || !tr->last_row || !tr->x || !tr->y || !tr->z_rel ||
                             !tr->time_ref || !tr->sin_phi || !tr->dzds || !tr->q_pt)) return TPC_EINVAL;
  const MergeLayout L = merge_layout(t->geom, tr->max_tracks);
  if (!t->params.arena || L.total > t->params.arena_bytes) return TPC_ENOMEM;
  if (L.n_cells + 1 >= 2147483000ull) return TPC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* A = static_cast<char*>(t->params.arena);
  const int K = tr->max_tracks;
  MergeConsts c{};
  c.n_sectors = t->geom.n_sectors; c.n_rows = t->geom.n_rows; c.n_tcell = L.n_tcell;
  c.gap = mp->max_row_gap; c.overlap = mp->max_row_overlap; c.max_tracks = K;
  c.x0 = t->geom.x0_cm; c.pitch = t->geom.row_pitch_cm;
  c.Z = t->consts.Z; c.inv_Z = t->consts.inv_Z; c.cB = t->consts.cB; c.sin_phi_max = t->consts.sin_phi_max;
  c.cut_y = mp->cut_y_cm; c.cut_z = mp->cut_z_cm; c.cut_s = mp->cut_sin_phi; c.cut_k = mp->cut_q_pt;
  c.wy = (float)(1.0 / ((double)mp->cut_y_cm * (double)mp->cut_y_cm));
  c.wz = (float)(1.0 / ((double)mp->cut_z_cm * (double)mp->cut_z_cm));
  c.ws = (float)(1.0 / ((double)mp->cut_sin_phi * (double)mp->cut_sin_phi));
  c.wk = (float)(1.0 / ((double)mp->cut_q_pt * (double)mp->cut_q_pt));
  c.inv_cell = 1.0f / (float)kMergeCellTimeBins;
  c.t_window = (float)((double)mp->cut_z_cm / (double)t->geom.time_bin_cm + 0.5);
  c.xr = t->consts.xr;
  const MergeCeConsts ce{mp->cut_dzds, (float)(1.0 / ((double)mp->cut_dzds * (double)mp->cut_dzds))};
  MergeTracks T{tr->n_tracks, tr->seed_hit, tr->sector, tr->first_row, tr->last_row, tr->x, tr->y, tr->z_rel, tr->time_ref, tr->sin_phi, tr->dzds, tr->q_pt};
  MergeScratch S{reinterpret_cast<uint32_t*>(A + L.cell_start), reinterpret_cast<uint32_t*>(A + L.cell_cursor),
                 reinterpret_cast<uint32_t*>(A + L.cell_of), reinterpret_cast<uint32_t*>(A + L.cand_idx),
                 reinterpret_cast<float4*>(A + L.cand_a), reinterpret_cast<float2*>(A + L.cand_b),
                 reinterpret_cast<unsigned long long*>(A + L.out_key), reinterpret_cast<int32_t*>(A + L.out_b),
                 reinterpret_cast<unsigned long long*>(A + L.in_key)};
  float* out_t = reinterpret_cast<float*>(A + L.out_t);
  int64_t launches = 0;
  cudaMemsetAsync(out->n_links, 0, 4, st);
  if (K > 0) {
    cudaMemsetAsync(out->next, 0xFF, 4 * (size_t)K, st);
    cudaMemsetAsync(out->prev, 0xFF, 4 * (size_t)K, st);
    cudaMemsetAsync(out->t_ce, 0, 4 * (size_t)K, st);
    cudaMemsetAsync(S.cell_start, 0, 4 * (L.n_cells + 1), st);
    cudaMemsetAsync(S.cell_cursor, 0, 4 * L.n_cells, st);
    cudaMemsetAsync(S.in_key, 0xFF, 8 * (size_t)K, st);
    const int g256 = (K + 255) / 256;
    k_merge_cell_count<<<g256, 256, 0, st>>>(T, S, c); ++launches;
    launches += exclusive_scan_u32(S.cell_start, S.cell_start, L.n_cells + 1, reinterpret_cast<uint32_t*>(A + L.scan), st);
    k_merge_cell_fill<<<g256, 256, 0, st>>>(T, S, c); ++launches;
    k_merge_ce_match<<<(K + kMergeThreads - 1) / kMergeThreads, kMergeThreads, 0, st>>>(T, S, out_t, c, ce); ++launches;
    k_merge_ce_link<<<g256, 256, 0, st>>>(T, S, out_t, out->next, out->prev, out->t_ce, out->n_links, c); ++launches;
  }
  t->last_merge_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C8: refit of the chains linked by C7 (merge.cuh) ----
int tpc_refit_chains(tpc_tracker_t* t, const tpc_tracks_t* tr, const tpc_merged_t* mg, void* cuda_stream, tpc_refit_t* out) {
  if (!t || !tr || !mg || !out) return TPC_EINVAL;
  if (tr->max_tracks < 0 || !tr->n_tracks || !out->ok || !out->chain_hits || !out->chain_pieces || !out->par7 || !out->cov9) return TPC_EINVAL;
  if (tr->max_tracks > 0 && (!tr->hit_y_time || !tr->hit_row || !tr->sector || !tr->n_hits || !tr->hit_offset || !tr->x ||
                             !tr->y || !tr->z_rel || !tr->time_ref || !tr->sin_phi || !tr->dzds || !tr->q_pt || !mg->next || !mg->prev)) return TPC_EINVAL;
  const int K = tr->max_tracks;
  const size_t need = 512 + 4 * (size_t)std::max(K, 1);
  if (!t->params.arena || need > t->params.arena_bytes) return TPC_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* A = static_cast<char*>(t->params.arena);
  uint32_t* n_roots = reinterpret_cast<uint32_t*>(A);
  uint32_t* work_counter = reinterpret_cast<uint32_t*>(A + 256);
  uint32_t* root_list = reinterpret_cast<uint32_t*>(A + 512);
  MergeConsts c{};
  c.n_sectors = t->geom.n_sectors; c.n_rows = t->geom.n_rows; c.max_tracks = K;
  {
    const double T = (double)t->geom.tan_half_sector;
    c.Cd = (float)((1.0 - T * T) / (1.0 + T * T));
    c.Sd = (float)(2.0 * T / (1.0 + T * T));
  }
  MergeTracks T{tr->n_tracks, tr->seed_hit, tr->sector, tr->first_row, tr->last_row, tr->x, tr->y, tr->z_rel, tr->time_ref, tr->sin_phi, tr->dzds, tr->q_pt};
  RefitIo io{reinterpret_cast<const float2*>(tr->hit_y_time), tr->hit_row, tr->n_hits, tr->hit_offset, tr->max_track_hits, mg->next, mg->prev,
             out->ok, out->chain_hits, out->chain_pieces, out->par7, out->cov9};
  int64_t launches = 0;
  cudaMemsetAsync(n_roots, 0, 512, st);
  if (K > 0) {
    k_refit_roots<<<(K + 255) / 256, 256, 0, st>>>(T, io, root_list, n_roots, c); ++launches;
    k_refit_chains<<<std::min(t->ctas_refit, (K + kMergeThreads - 1) / kMergeThreads), kMergeThreads, 0, st>>>(T, io, root_list, n_roots, work_counter, c, t->consts); ++launches;
  }
  t->last_merge_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C12: refit of every chain root with the full covariance and the material of the gas (fullfit.cuh) ----
int tpc_refit_full(tpc_tracker_t* t, const tpc_fullfit_params_t* fp, const tpc_tracks_t* tr, const tpc_merged_t* mg, void* cuda_stream,
                   tpc_fullfit_t* out) {
  return tpc_refit_full_ce(t, fp, tr, mg, nullptr, cuda_stream, out);
}

int tpc_refit_full_ce(tpc_tracker_t* t, const tpc_fullfit_params_t* fp, const tpc_tracks_t* tr, const tpc_merged_t* mg, const tpc_ce_merged_t* ce,
                      void* cuda_stream, tpc_fullfit_t* out) {
  if (!t || !fp || !tr || !mg || !out) return TPC_EINVAL;
  if (!(fp->inv_x0_per_cm >= 0 && fp->dedx_mip_gev_per_cm >= 0 && fp->mass_gev >= 0 && fp->eloss_sigma >= 0)) return TPC_EINVAL;
  if (tr->max_tracks < 0 || !tr->n_tracks || !out->ok || !out->chain_hits || !out->chain_pieces || !out->par7 || !out->cov15) return TPC_EINVAL;
  if (tr->max_tracks > 0 && (!tr->hit_y_time || !tr->hit_row || !tr->sector || !tr->n_hits || !tr->hit_offset || !tr->x ||
                             !tr->y || !tr->z_rel || !tr->time_ref || !tr->sin_phi || !tr->dzds || !tr->q_pt || !mg->next || !mg->prev)) return TPC_EINVAL;
  const int K = tr->max_tracks;
  const size_t need = 512 + 4 * (size_t)std::max(K, 1);
  if (!t->params.arena || need > t->params.arena_bytes) return TPC_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  char* A = static_cast<char*>(t->params.arena);
  uint32_t* n_roots = reinterpret_cast<uint32_t*>(A);
  uint32_t* work_counter = reinterpret_cast<uint32_t*>(A + 256);
  uint32_t* root_list = reinterpret_cast<uint32_t*>(A + 512);
  MergeConsts c{};
  c.n_sectors = t->geom.n_sectors; c.n_rows = t->geom.n_rows; c.max_tracks = K;
  {
    const double T = (double)t->geom.tan_half_sector;
    c.Cd = (float)((1.0 - T * T) / (1.0 + T * T));
    c.Sd = (float)(2.0 * T / (1.0 + T * T));
  }
  FullFitConsts m{};                                   // constants derived in double, rounded once
  m.inv_x0 = fp->inv_x0_per_cm; m.dedx_mip = fp->dedx_mip_gev_per_cm; m.eloss_sigma = fp->eloss_sigma;
  m.m2 = (float)((double)fp->mass_gev * (double)fp->mass_gev);
  m.ms2 = (float)(13.6e-3 * 13.6e-3);                  // Highland: 13.6 MeV, in GeV
  MergeTracks T{tr->n_tracks, tr->seed_hit, tr->sector, tr->first_row, tr->last_row, tr->x, tr->y, tr->z_rel, tr->time_ref, tr->sin_phi, tr->dzds, tr->q_pt};
  if (ce && tr->max_tracks > 0 && (!ce->next || !ce->prev || !ce->t_ce)) return TPC_EINVAL;
  FullFitIo io{reinterpret_cast<const float2*>(tr->hit_y_time), tr->hit_row, tr->n_hits, tr->hit_offset, tr->max_track_hits, mg->next, mg->prev,
               ce ? ce->next : nullptr, ce ? ce->prev : nullptr, ce ? ce->t_ce : nullptr,
               out->ok, out->chain_hits, out->chain_pieces, out->par7, out->cov15};
  int64_t launches = 0;
  cudaMemsetAsync(n_roots, 0, 512, st);
  if (K > 0) {
    k_fullfit_roots<<<(K + 255) / 256, 256, 0, st>>>(T, io, root_list, n_roots, c); ++launches;
    k_refit_full<<<std::min(t->ctas_fullfit, (K + kMergeThreads - 1) / kMergeThreads), kMergeThreads, 0, st>>>(T, io, root_list, n_roots, work_counter, c, t->consts, m); ++launches;
  }
  t->last_merge_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C11: track-based hit rejection + track-model residual coding (compress.cuh) ----
int tpc_compress_tracks(tpc_tracker_t* t, const tpc_compress_params_t* cp, const tpc_tracks_t* tr, int64_t n_clusters, void* cuda_stream,
                        tpc_compressed_t* out) {
  if (!t || !cp || !tr || !out || n_clusters < 0) return TPC_EINVAL;
  if (!(cp->reject_q_pt > 0 && cp->step_y_cm > 0 && cp->step_z_cm > 0)) return TPC_EINVAL;
  if (tr->max_tracks < 0 || tr->max_track_hits < 0 || !tr->n_tracks || !out->ok || (n_clusters > 0 && !out->reject)) return TPC_EINVAL;
  if (tr->max_track_hits > 0 && (!out->res_y || !out->res_z)) return TPC_EINVAL;
  if (tr->max_tracks > 0 && (!tr->hit_y_time || !tr->hit_row || !tr->hit_index || !tr->n_hits || !tr->hit_offset || !tr->x || !tr->y || !tr->z_rel ||
                             !tr->time_ref || !tr->sin_phi || !tr->dzds || !tr->q_pt || !tr->cov9)) return TPC_EINVAL;
  if (!t->params.arena || t->params.arena_bytes < 256) return TPC_ENOMEM;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  uint32_t* work_counter = reinterpret_cast<uint32_t*>(t->params.arena);
  const int K = tr->max_tracks;
  CompressIo io{tr->n_tracks, K, tr->max_track_hits, tr->n_hits, tr->hit_offset, tr->hit_index, reinterpret_cast<const float2*>(tr->hit_y_time), tr->hit_row,
                tr->x, tr->y, tr->z_rel, tr->sin_phi, tr->dzds, tr->q_pt, tr->time_ref, tr->cov9,
                out->reject, out->ok, out->res_y, out->res_z, cp->reject_q_pt, cp->step_y_cm, cp->step_z_cm};
  int64_t launches = 0;
  cudaMemsetAsync(work_counter, 0, 256, st);
  if (n_clusters > 0) cudaMemsetAsync(out->reject, 0, (size_t)n_clusters, st);
  if (K > 0) {
    k_compress_reject<<<(int)(((int64_t)K * 32 + 255) / 256), 256, 0, st>>>(io); ++launches;
    k_compress_tracks<<<std::min(t->ctas_refit, (K + kMergeThreads - 1) / kMergeThreads), kMergeThreads, 0, st>>>(io, work_counter, t->consts); ++launches;
  }
  t->last_merge_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}


// ---- C9: beam-line time / offset of every state in par7 (merge.cuh) ----
int tpc_vertex_time(tpc_tracker_t* t, const int32_t* n_tracks, int32_t max_tracks, const float* par7, void* cuda_stream,
                    int32_t* ok, float* vertex_time, float* vertex_y) {
  if (!t || !n_tracks || max_tracks < 0 || !ok || !vertex_time || !vertex_y || (max_tracks > 0 && !par7)) return TPC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (max_tracks > 0)
    k_vertex_time<<<(max_tracks + 255) / 256, 256, 0, st>>>(n_tracks, max_tracks, par7, ok, vertex_time, vertex_y, t->consts.Z, t->consts.cB,
                                                          t->consts.sin_phi_max);
  t->last_merge_launches = max_tracks > 0 ? 1 : 0;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}

int64_t tpc_merge_last_launches(const tpc_tracker_t* t) { return t ? t->last_merge_launches : -1; }

int tpc_tracker_destroy(tpc_tracker_t* t) {
  if (!t) return TPC_EINVAL;
  for (int i = 0; i <= N_STEPS; ++i) if (t->ev[i]) cudaEventDestroy(t->ev[i]);
  if (t->tables) cudaFree(t->tables);
  delete t;
  return TPC_OK;
}

int tpc_tracker_arena_plan(const tpc_tracker_t* t, int32_t i, const char** name, size_t* offset, size_t* bytes,
                           int32_t* first_step, int32_t* last_step) {
  if (!t) return -1;
  const auto& a = t->plan.allocs();
  if (i < 0 || i >= (int)a.size()) return -1;
  if (name) *name = a[i].name.c_str();
  if (offset) *offset = a[i].offset;
  if (bytes) *bytes = a[i].bytes;
  if (first_step) *first_step = a[i].first_step;
  if (last_step) *last_step = a[i].last_step;
  return (int)a.size();
}

int64_t tpc_tracker_last_launches(const tpc_tracker_t* t) { return t ? t->last_launches : -1; }

int tpc_tracker_work_counters(tpc_tracker_t* t, void* cuda_stream, int64_t* out, int32_t capacity) {
  if (!t || !out || capacity < 0) return TPC_EINVAL;
  struct { int32_t i32[8]; unsigned long long u64[28]; } h;     // the 256-byte counter block
  static_assert(sizeof(h) == 256, "counter block");
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (cudaMemcpyAsync(&h, t->counters, 256, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  int64_t v[22] = {h.i32[kCntTracklets], h.i32[kCntStartHits], (int64_t)(uint32_t)h.i32[kCntInvalid], 0, 0, 0};
  for (int ph = 0; ph < 4; ++ph)
    for (int k = 0; k < 3; ++k) {
      v[6 + 3 * ph + k] = (int64_t)h.u64[kCnt64Phase0 - 4 + 3 * ph + k];
      v[3 + k] += v[6 + 3 * ph + k];
    }
  for (int k = 0; k < 4; ++k) v[18 + k] = (int64_t)h.u64[kCnt64Rare0 - 4 + k];
  for (int i = 0; i < 22 && i < capacity; ++i) out[i] = v[i];
  return 22;
}

int tpc_tracker_step_ms(tpc_tracker_t* t, float* ms_out, int32_t capacity) {
  if (!t || !ms_out) return TPC_EINVAL;
  if (!t->profile || !t->have_times) return TPC_EINVAL;
  if (cudaEventSynchronize(t->ev[N_STEPS]) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  for (int i = 0; i < N_STEPS && i < capacity; ++i)
    if (cudaEventElapsedTime(&ms_out[i], t->ev[i], t->ev[i + 1]) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  return N_STEPS;
}

int tpc_track_timeframe(tpc_tracker_t* t, const tpc_clusters_t* cl, int64_t n, void* cuda_stream, tpc_tracks_t* o) {
  if (!t || !cl || !o || n < 0 || n > t->cap.max_clusters) return TPC_EINVAL;
  if (n > 0 && (!cl->row || !cl->pad || !cl->time)) return TPC_EINVAL;
  if (!o->n_tracks || !o->n_track_hits || !o->status || o->max_tracks < 0 || o->max_track_hits < 0) return TPC_EINVAL;
  if (o->max_tracks > 0 && (!o->seed_hit || !o->sector || !o->first_row || !o->last_row || !o->n_hits || !o->hit_offset ||
                            !o->x || !o->y || !o->z_rel || !o->time_ref || !o->sin_phi || !o->dzds || !o->q_pt)) return TPC_EINVAL;
  if (o->max_track_hits > 0 && !o->hit_index) return TPC_EINVAL;
  const bool link_taps = o->link_up || o->link_down || o->is_start_hit;
  if (link_taps && !(o->link_up && o->link_down && o->is_start_hit)) return TPC_EINVAL;
  const bool tl_taps = o->tracklet_seed || o->tracklet_n_hits || o->tracklet_row_hit || o->tracklet_par || o->n_tracklets;
  if (tl_taps && o->max_tracklets < 0) return TPC_EINVAL;

  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const Consts& c = t->consts;
  const ArenaPlan& P = t->plan;
  const Ids& id = t->id;
  void* A = t->params.arena;
  const int T = (int)t->cap.max_tracklets;
  int64_t launches = 0;
  auto mark = [&](int step) { if (t->profile) cudaEventRecord(t->ev[step], st); };

  uint32_t* bin_start = P.ptr<uint32_t>(A, id.bin_start);
  uint32_t* sort_keys = P.ptr<uint32_t>(A, id.sort_keys);
  uint32_t* sort_hist = P.ptr<uint32_t>(A, id.sort_hist);
  float2* yt = P.ptr<float2>(A, id.yt);
  uint32_t* orig = P.ptr<uint32_t>(A, id.orig);
  uint16_t* hsr = P.ptr<uint16_t>(A, id.hsr);
  int* link_up = P.ptr<int>(A, id.link_up);
  int* link_down = P.ptr<int>(A, id.link_down);
  int* link_up_clean = P.ptr<int>(A, id.link_up_clean);
  uint8_t* start_flag = P.ptr<uint8_t>(A, id.start_flag);
  uint32_t* cell_count = P.ptr<uint32_t>(A, id.cell_count);
  uint32_t* start_hits = P.ptr<uint32_t>(A, id.start_hits);
  uint2* chunks = P.ptr<uint2>(A, id.chunks);
  int32_t* counters = t->counters;                             // layout: kCnt* in tracklet.cuh
  uint32_t* n_invalid = reinterpret_cast<uint32_t*>(counters + kCntInvalid);
  TrackletSeeds seeds;
  seeds.a = P.ptr<int4>(A, id.seeds_a);
  seeds.b = P.ptr<float4>(A, id.seeds_b);
  uint32_t* scan_a = P.ptr<uint32_t>(A, id.scan_a);
  uint32_t* scan_b = P.ptr<uint32_t>(A, id.scan_b);
  unsigned long long* claim = P.ptr<unsigned long long>(A, id.claim);
  uint32_t* owned = P.ptr<uint32_t>(A, id.owned);
  uint32_t* flag = P.ptr<uint32_t>(A, id.flag);
  uint32_t* track_idx = P.ptr<uint32_t>(A, id.track_idx);
  uint32_t* hit_off = P.ptr<uint32_t>(A, id.hit_off);
  uint32_t* track_slot = P.ptr<uint32_t>(A, id.track_slot);
  TrackletStore tl;
  tl.row_hit = P.ptr<int>(A, id.row_hit);
  tl.meta = P.ptr<int4>(A, id.tl_meta);
  tl.rec = P.ptr<float4>(A, id.tl_rec);
  tl.cur = P.ptr<float4>(A, id.tl_cur);
  tl.cap = (size_t)T;

  const int hit_ctas = (int)std::max<int64_t>((n + 255) / 256, 1);
  const int link_ctas = (int)std::max<int64_t>((n + kLinkThreads - 1) / kLinkThreads, 1);

  // ---- C1 ingest: stable LSD radix sort on the grid bin index, then the bin offsets ----
  mark(S_SORT);
  cudaMemsetAsync(counters, 0, 256, st);
  if (link_taps && n > 0) {
    cudaMemsetAsync(o->link_up, 0xFF, 4 * (size_t)n, st);
    cudaMemsetAsync(o->link_down, 0xFF, 4 * (size_t)n, st);
    cudaMemsetAsync(o->is_start_hit, 0, (size_t)n, st);
  }
  if (n > 0) {
    const int n_tiles = (int)((n + kRadixTile - 1) / kRadixTile);
    const int passes = t->cap.sort_passes, dbits = t->cap.sort_digit_bits;
    const uint32_t mask = (1u << dbits) - 1u;
    RadixDst fin{sort_keys, orig, yt};
    RadixDst tmp{P.ptr<uint32_t>(A, id.tmp_keys), P.ptr<uint32_t>(A, id.tmp_orig), P.ptr<float2>(A, id.tmp_yt)};
    RadixSrc src{cl->row, cl->pad, cl->time, nullptr, nullptr, nullptr};
    for (int p = 0; p < passes; ++p) {
      const RadixDst dst = ((passes - 1 - p) % 2 == 0) ? fin : tmp;
      const size_t hist_n = (size_t)(mask + 1) * n_tiles;
      if (p == 0) k_radix_histogram<true><<<n_tiles, kRadixThreads, 0, st>>>(src, n, p * dbits, mask, sort_hist, n_tiles, c);
      else k_radix_histogram<false><<<n_tiles, kRadixThreads, 0, st>>>(src, n, p * dbits, mask, sort_hist, n_tiles, c);
      ++launches;
      launches += exclusive_scan_u32(sort_hist, sort_hist, hist_n, scan_a, st);
      if (p == 0) k_radix_scatter<true><<<n_tiles, kRadixThreads, kRadixScatterSmem, st>>>(src, dst, n, p * dbits, mask, sort_hist, n_tiles, n_invalid, c);
      else k_radix_scatter<false><<<n_tiles, kRadixThreads, kRadixScatterSmem, st>>>(src, dst, n, p * dbits, mask, sort_hist, n_tiles, n_invalid, c);
      ++launches;
      src = RadixSrc{nullptr, nullptr, nullptr, dst.keys, dst.orig, dst.yt};
    }
  }
  mark(S_GRID);
  {
    uint4* gap_list = P.ptr<uint4>(A, id.gap_list);
    uint32_t* n_gaps = reinterpret_cast<uint32_t*>(counters + kCntGridGaps);
    k_grid_build<<<(int)((n + 1 + 255) / 256), 256, 0, st>>>(sort_keys, n, bin_start, hsr, gap_list, n_gaps, c); ++launches;
    k_grid_fill_gaps<<<148 * 8, 256, 0, st>>>(gap_list, n_gaps, bin_start); ++launches;
  }

  // ---- C2 neighbours finder ----
  mark(S_FINDER);
  k_neighbours_finder<<<hit_ctas, kFinderThreads, 0, st>>>(yt, orig, hsr, bin_start, link_up, link_down, c); ++launches;

  // ---- C3 cleaner + C4 start hits ----
  mark(S_CLEAN_START);
  k_clean_links_find_starts<<<link_ctas, kLinkThreads, 0, st>>>(link_up, link_down, bin_start, link_up_clean, start_flag,
                                                                orig, link_taps ? o->link_up : nullptr, o->link_down,
                                                                o->is_start_hit, c); ++launches;
  mark(S_COMPACT);
  {
    const StartCells sc{t->cap.n_slices, t->cap.slice_bins, (uint32_t)t->cap.n_cells};
    const int cell_ctas = (int)((t->cap.n_cells + kLinkThreads - 1) / kLinkThreads);
    const size_t n_cells = (size_t)t->cap.n_cells;
    k_start_cell_count<<<cell_ctas, kLinkThreads, 0, st>>>(start_flag, bin_start, sc, cell_count, c); ++launches;
    launches += exclusive_scan_u32(cell_count, cell_count, n_cells, scan_a, st);
    k_start_cell_write<<<cell_ctas, kLinkThreads, 0, st>>>(start_flag, bin_start, sc, cell_count, scan_a + scan_tiles(n_cells), start_hits,
                                                           (uint32_t)T, counters, c); ++launches;
    if (t->follow_rows) {    // work units of the row-synchronous follower: <= kFrChunk tracklets of one (sector, slice) group each
      k_follow_chunk_list<<<1, kScanThreads, 0, st>>>(cell_count, scan_a + scan_tiles(n_cells), t->geom.n_sectors * t->cap.n_slices, c.n_rows,
                                                      chunks, counters); ++launches;
    }
  }

  // ---- C5 tracklet constructor ----
  mark(S_TL_INIT);
  const int64_t tl_bound = std::min<int64_t>(T, n / std::max(2, c.seed_min_hits) + 1);   // start hits own disjoint chains
  k_tracklet_init<<<(int)((tl_bound + 255) / 256), 256, 0, st>>>(yt, hsr, link_up_clean, start_hits, counters, seeds, tl.row_hit, c); ++launches;
  {
    const int need = (int)((tl_bound + kTrackletThreads - 1) / kTrackletThreads);
    const int64_t rows_need = std::max<int64_t>(1, std::min<int64_t>(t->cap.max_chunks, tl_bound / kFrChunk + (int64_t)t->geom.n_sectors * t->cap.n_slices + 1));
    mark(S_FIT_UP);
    k_tracklet_fit<false><<<std::min(t->ctas_fit_up, need), kTrackletThreads, 0, st>>>(yt, orig, seeds, counters, tl, c);
    mark(S_FOLLOW_UP);
    if (t->follow_rows) k_follow_rows<false><<<(int)std::min<int64_t>(t->ctas_rows_up, rows_need), kFrThreads, sizeof(FrSmem), st>>>(yt, orig, bin_start, seeds, counters, chunks, tl, c);
    else k_tracklet_follow<false><<<std::min(t->ctas_follow_up, need), kTrackletThreads, 0, st>>>(yt, orig, bin_start, seeds, counters, tl, c);
    mark(S_FIT_DOWN);
    k_tracklet_fit<true><<<std::min(t->ctas_fit_down, need), kTrackletThreads, 0, st>>>(yt, orig, seeds, counters, tl, c);
    mark(S_FOLLOW_DOWN);
    if (t->follow_rows) k_follow_rows<true><<<(int)std::min<int64_t>(t->ctas_rows_down, rows_need), kFrThreads, sizeof(FrSmem), st>>>(yt, orig, bin_start, seeds, counters, chunks, tl, c);
    else k_tracklet_follow<true><<<std::min(t->ctas_follow_down, need), kTrackletThreads, 0, st>>>(yt, orig, bin_start, seeds, counters, tl, c);
    launches += 4;
  }
  const int warp_ctas = (int)((tl_bound * 32 + kSelectorThreads - 1) / kSelectorThreads);
  if (tl_taps) {
    k_export_tracklets<<<warp_ctas, kSelectorThreads, 0, st>>>(tl, counters, orig, o->n_tracklets, o->tracklet_seed, o->tracklet_n_hits,
                                                               o->tracklet_row_hit, o->tracklet_par, o->max_tracklets, c); ++launches;
  }

  // ---- C6 tracklet selector ----
  mark(S_CLAIM);
  if (n > 0) cudaMemsetAsync(claim, 0, 8 * (size_t)n, st);
  k_selector_claim_top<<<(int)((tl_bound + 255) / 256), 256, 0, st>>>(tl, counters, claim, c); ++launches;
  k_selector_claim<<<warp_ctas, kSelectorThreads, 0, st>>>(tl, counters, claim, c); ++launches;
  mark(S_COUNT);
  cudaMemsetAsync(owned, 0, 4 * (size_t)T, st);
  k_selector_count_hits<<<hit_ctas, 256, 0, st>>>(claim, bin_start, owned, c); ++launches;
  k_selector_flag<<<(T + 255) / 256, 256, 0, st>>>(owned, flag, T, c); ++launches;
  mark(S_SELECT_SCAN);
  launches += exclusive_scan_u32(flag, track_idx, (size_t)T, scan_a, st);
  launches += exclusive_scan_u32(owned, hit_off, (size_t)T, scan_b, st);
  mark(S_EMIT);
  TrackOutputs to;
  to.max_tracks = o->max_tracks; to.max_track_hits = o->max_track_hits;
  to.n_tracks = o->n_tracks; to.n_track_hits = o->n_track_hits; to.status = o->status;
  to.seed_hit = o->seed_hit; to.sector = o->sector; to.first_row = o->first_row; to.last_row = o->last_row; to.n_hits = o->n_hits;
  to.hit_offset = o->hit_offset; to.x = o->x; to.y = o->y; to.z_rel = o->z_rel; to.time_ref = o->time_ref;
  to.sin_phi = o->sin_phi; to.dzds = o->dzds; to.q_pt = o->q_pt; to.cov9 = o->cov9; to.hit_index = o->hit_index;
  to.hit_yt = reinterpret_cast<float2*>(o->hit_y_time); to.hit_row = o->hit_row;
  const int n_scan_tiles = (int)scan_tiles((size_t)T);
  k_selector_map<<<(int)((tl_bound + 255) / 256), 256, 0, st>>>(counters, flag, track_idx, track_slot); ++launches;
  const int64_t emit_warps = std::max<int64_t>(std::min<int64_t>(tl_bound, o->max_tracks), 1);      // warp 0 also writes the scalars
  k_selector_emit<<<(int)((emit_warps * 32 + kSelectorThreads - 1) / kSelectorThreads), kSelectorThreads, 0, st>>>(
      tl, counters, claim, track_slot, hit_off, scan_a + n_scan_tiles, scan_b + n_scan_tiles, orig, yt, hsr, start_hits, n_invalid, to, c); ++launches;
  mark(N_STEPS);
  t->have_times = t->profile;
  t->last_launches = launches;
  if (cudaGetLastError() != cudaSuccess) return TPC_ECUDA;
  return TPC_OK;
}

int tpc_selftest_fast_math(void* cuda_stream, uint64_t* mismatches_out) {
  if (!mismatches_out) return TPC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  unsigned long long* d = nullptr;
  if (cudaMalloc(&d, 16) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  unsigned long long h[2] = {0, 0};
  bool ok = cudaMemsetAsync(d, 0, 16, st) == cudaSuccess;
  if (ok) { k_selftest_fast_math<<<148 * 16, 256, 0, st>>>(d); ok = cudaGetLastError() == cudaSuccess; }
  ok = ok && cudaMemcpyAsync(h, d, 16, cudaMemcpyDeviceToHost, st) == cudaSuccess && cudaStreamSynchronize(st) == cudaSuccess;
  cudaFree(d);
  if (!ok) { cudaGetLastError(); return TPC_ECUDA; }
  mismatches_out[0] = h[0]; mismatches_out[1] = h[1];
  return TPC_OK;
}

int tpc_selftest_alu_peak(void* cuda_stream, double* out) {
  if (!out) return TPC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int ctas = sms * 8 * 4;                        // 4 waves of 8 resident CTAs of 256 threads per SM
  float* sink = nullptr;
  cudaEvent_t e[3] = {};
  bool ok = cudaMalloc(&sink, (size_t)ctas * 4) == cudaSuccess;
  for (int i = 0; i < 3 && ok; ++i) ok = cudaEventCreate(&e[i]) == cudaSuccess;
  float ms[2] = {0.0f, 0.0f};
  if (ok) {
    k_alu_peak_scalar<<<ctas, 256, 0, st>>>(sink, 1.0000001f, 1.0e-9f);     // warm-up (clocks, instruction cache)
    k_alu_peak_packed<<<ctas, 256, 0, st>>>(sink, 1.0000001f, 1.0e-9f);
    cudaEventRecord(e[0], st);
    k_alu_peak_scalar<<<ctas, 256, 0, st>>>(sink, 1.0000001f, 1.0e-9f);
    cudaEventRecord(e[1], st);
    k_alu_peak_packed<<<ctas, 256, 0, st>>>(sink, 1.0000001f, 1.0e-9f);
    cudaEventRecord(e[2], st);
    ok = cudaStreamSynchronize(st) == cudaSuccess && cudaEventElapsedTime(&ms[0], e[0], e[1]) == cudaSuccess &&
         cudaEventElapsedTime(&ms[1], e[1], e[2]) == cudaSuccess && cudaGetLastError() == cudaSuccess;
  }
  for (int i = 0; i < 3; ++i) if (e[i]) cudaEventDestroy(e[i]);
  if (sink) cudaFree(sink);
  if (!ok || ms[0] <= 0.0f || ms[1] <= 0.0f) { cudaGetLastError(); return TPC_ECUDA; }
  const double lane_inst = (double)ctas * 256.0 * (double)kAluIters * (double)(2 * kAluChains);
  out[0] = lane_inst / ((double)ms[0] * 1.0e-3);
  out[1] = 2.0 * lane_inst / ((double)ms[1] * 1.0e-3);
  return TPC_OK;
}

int tpc_track_timeframe_host(tpc_tracker_t* t, const tpc_clusters_t* hc, int64_t n, void* cuda_stream, tpc_tracks_t* ho) {
  if (!t || !hc || !ho || n < 0 || n > t->cap.max_clusters) return TPC_EINVAL;
  if (t->id.stage_in < 0) return TPC_EINVAL;
  if (n > 0 && (!hc->row || !hc->pad || !hc->time)) return TPC_EINVAL;
  if (!ho->n_tracks || !ho->n_track_hits || !ho->status) return TPC_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  void* A = t->params.arena;
  const size_t N = (size_t)t->cap.max_clusters;
  float* d_in = t->plan.ptr<float>(A, t->id.stage_in);
  const int64_t K = std::min<int64_t>(t->cap.max_tracks, ho->max_tracks);
  const int64_t H = std::min<int64_t>(t->cap.max_track_hits, ho->max_track_hits);
  // carve the output staging block
  char* p = t->plan.ptr<char>(A, t->id.stage_out);
  auto take = [&](size_t bytes) { char* q = p; p += (bytes + 15) / 16 * 16; return q; };
  tpc_tracks_t d;
  std::memset(&d, 0, sizeof(d));
  d.max_tracks = (int32_t)K; d.max_track_hits = H;
  d.n_track_hits = reinterpret_cast<int64_t*>(take(8));
  d.n_tracks = reinterpret_cast<int32_t*>(take(4));
  d.status = reinterpret_cast<int32_t*>(take(4));
  d.hit_offset = reinterpret_cast<int64_t*>(take(8 * (size_t)K));
  int32_t** i32s[] = {&d.seed_hit, &d.sector, &d.first_row, &d.last_row, &d.n_hits};
  for (auto pp : i32s) *pp = reinterpret_cast<int32_t*>(take(4 * (size_t)K));
  float** f32s[] = {&d.x, &d.y, &d.z_rel, &d.time_ref, &d.sin_phi, &d.dzds, &d.q_pt};
  for (auto pp : f32s) *pp = reinterpret_cast<float*>(take(4 * (size_t)K));
  d.cov9 = ho->cov9 ? reinterpret_cast<float*>(take(36 * (size_t)K)) : nullptr;
  d.hit_index = reinterpret_cast<int32_t*>(take(4 * (size_t)H));

  tpc_clusters_t dc;
  dc.row = d_in; dc.pad = d_in + N; dc.time = d_in + 2 * N; dc.charge = nullptr;
  if (n > 0) {
    if (cudaMemcpyAsync(d_in, hc->row, 4 * (size_t)n, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d_in + N, hc->pad, 4 * (size_t)n, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(d_in + 2 * N, hc->time, 4 * (size_t)n, cudaMemcpyHostToDevice, st) != cudaSuccess) {
      cudaGetLastError(); return TPC_ECUDA;
    }
  }
  // Frames in flight on several handles / streams (double buffering): their COPIES should overlap the kernels of another
  // frame, their KERNELS should not overlap each other -- two constructors running side by side halve each other's L2 (the
  // follower lives on a 77 % L2 hit rate) and finish later than one after the other.  A process-wide event chain orders the
  // compute sections of all host-entry calls; the copies before and after stay unordered.
  static std::mutex compute_mutex;
  static cudaEvent_t compute_done = nullptr;
  int rc;
  {
    std::lock_guard<std::mutex> lock(compute_mutex);
    if (!compute_done) { if (cudaEventCreateWithFlags(&compute_done, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); compute_done = nullptr; } }
    else cudaStreamWaitEvent(st, compute_done, 0);
    rc = tpc_track_timeframe(t, &dc, n, cuda_stream, &d);
    if (compute_done) cudaEventRecord(compute_done, st);
  }
  if (rc != TPC_OK) return rc;
  struct { int64_t nh; int32_t nt; int32_t status; } head;
  if (cudaMemcpyAsync(&head.nh, d.n_track_hits, 8, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaMemcpyAsync(&head.nt, d.n_tracks, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaMemcpyAsync(&head.status, d.status, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  *ho->n_tracks = head.nt; *ho->n_track_hits = head.nh; *ho->status = head.status;
  const size_t k = (size_t)std::min<int64_t>(head.nt, K), h = (size_t)std::min<int64_t>(head.nh, H);
  bool ok = true;
  auto back = [&](void* dst, const void* src, size_t bytes) {
    if (dst && bytes) ok = ok && cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  };
  back(ho->hit_offset, d.hit_offset, 8 * k);
  back(ho->seed_hit, d.seed_hit, 4 * k); back(ho->sector, d.sector, 4 * k); back(ho->first_row, d.first_row, 4 * k);
  back(ho->last_row, d.last_row, 4 * k); back(ho->n_hits, d.n_hits, 4 * k);
  back(ho->x, d.x, 4 * k); back(ho->y, d.y, 4 * k); back(ho->z_rel, d.z_rel, 4 * k); back(ho->time_ref, d.time_ref, 4 * k);
  back(ho->sin_phi, d.sin_phi, 4 * k); back(ho->dzds, d.dzds, 4 * k); back(ho->q_pt, d.q_pt, 4 * k);
  if (d.cov9) back(ho->cov9, d.cov9, 36 * k);
  back(ho->hit_index, d.hit_index, 4 * h);
  if (!ok || cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return TPC_ECUDA; }
  return TPC_OK;
}

}  // extern "C"
