// C5 track following, row-synchronous form (BASELINE.json L5 item 4: "extrapolates row by row, with a ... grid search and
// shared-memory-staged row data"; the fit and the hit attachment are what costs compute).
//
// The per-lane follower (tracklet.cuh::k_tracklet_follow) lets every lane walk its own tracklet: two dependent global
// round trips per row step (grid offsets, then candidates), lane refill logic, 24 of 32 lanes busy.  Here a CTA owns a
// CHUNK of up to kFrChunk tracklets that start in the same (sector, time slice) and sweeps the pad rows in lock step:
//   * the tracklet states live in shared memory (64 bytes each); every row the still-active tracklets are re-compacted
//     onto consecutive lanes (an index list), so warps are full and no lane waits for a refill;
//   * the grid is time-major inside a sector-row (common.cuh::grid_bin), so everything the chunk can touch in pad row r --
//     the grid offsets and the (y, time) pairs of the time range its tracklets predict -- is ONE contiguous span each.
//     They are staged into shared memory by two bulk copies (cp.async.bulk + mbarrier complete_tx), the offsets three
//     rows and the hits two rows ahead of use, from the time range the tracklets themselves predict (linear
//     extrapolation of each state; tracklets that join in the next rows contribute from a per-row table);
//   * the window search then runs on shared memory.  A tracklet whose window is not covered by the staged range (a
//     wrong prediction, a range cut to the stage capacity, an exact distance tie) takes search_row_global(): the same
//     definition evaluated in global memory.  The staging is a prefetch hint only -- it never decides anything.
// Arithmetic per tracklet (transport, window, search predicate, update) is the same statement list as before, so the
// results are bit-identical to the per-lane follower and to the oracle.
#pragma once
#include "common.cuh"
#include "scan.cuh"
#include "tracklet.cuh"

namespace tpc {

#ifndef TPC_FR_CHUNK
#define TPC_FR_CHUNK 768
#endif
#ifndef TPC_FR_WARPS
#define TPC_FR_WARPS 11
#endif
#ifndef TPC_FR_BINS_CAP
#define TPC_FR_BINS_CAP 1536
#endif
#ifndef TPC_FR_HITS_CAP
#define TPC_FR_HITS_CAP 768
#endif
#ifndef TPC_FR_MIN_CTAS
#define TPC_FR_MIN_CTAS 2
#endif
constexpr int kFrChunk = TPC_FR_CHUNK;         // tracklets per work unit (one CTA at a time)
constexpr int kFrWorkers = TPC_FR_WARPS * 32;  // threads that follow tracklets
constexpr int kFrThreads = kFrWorkers + 32;    // + one warp whose lane 0 requests the bulk copies (off the workers' critical path)
constexpr int kFrBinStages = 4;                // grid offsets of the row used at step it + 3 are requested at step it
constexpr int kFrHitStages = 3;                // hits of the row used at step it + 2 are requested at step it
constexpr int kFrBinsCap = TPC_FR_BINS_CAP;    // uint32 entries per offsets stage
constexpr int kFrHitsCap = TPC_FR_HITS_CAP;    // float2 entries per hits stage
constexpr int kFrJoinRows = kRowStride + 8;    // per-row range table of the joining tracklets, index = row + 4
static_assert(kFrChunk <= 65535 && kFrChunk % 32 == 0, "chunk shape");

struct FrBinStage { int gb0, ngb, off, pad_; };   // first staged grid time bin, number of them, index of its first entry in the stage
struct FrHitStage { uint32_t lo, n; };            // sorted-hit index of the first staged hit, number of staged hits

struct FrSmem {
  float4 state[4][kFrChunk];                   // the tracklet record layout: (x, y, z, s) (t, k, c0, c1) (c2, c3, c4, c5) (d0, d1, d2, tstart)
  float2 hits[kFrHitStages][kFrHitsCap];
  uint32_t bins[kFrBinStages][kFrBinsCap];
  unsigned long long bar_bins[kFrBinStages], bar_hits[kFrHitStages];
  uint32_t packed[kFrChunk];                   // misses | row of the last update << 8 | hits << 16 | outermost row with a hit << 24
  uint16_t list[2][kFrChunk];                  // tracklets (slots) that survived the previous step / survive this one
  uint16_t join_sorted[kFrChunk];              // active slots ordered by their first target row
  int join_off[kRowStride + 2];                // first entry of a row in join_sorted
  int join_cnt[kRowStride + 2];
  uint8_t first_row[kFrChunk];                 // first target row of a slot, 255 = never active
  uint8_t r_init[kFrChunk];                    // row of the state the phase starts from
  int join_lo[kFrJoinRows], join_hi[kFrJoinRows];
  float xr[kRowStride], yoff[kRowStride], pscale[kRowStride];
  FrBinStage bst[kFrBinStages];
  FrHitStage hst[kFrHitStages];
  int n_list[3];                               // survivors: step it reads [it % 3], appends to [(it + 1) % 3]
  int acc_lo[2], acc_hi[2];                    // predicted grid-time-bin range of the row three steps ahead, by step parity
  int r_first, r_last_join, chunk;
};

// ---- mbarrier / bulk-copy primitives (sm_90+; SASS: SYNCS.*, UBLKCP) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared; both addresses 16-byte aligned, bytes a multiple of 16.
__device__ __forceinline__ void bulk_copy_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ float4 lds128_volatile(const float4* p) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(smem_u32(p)));
  return v;
}

// ---- work units: chunks of <= kFrChunk tracklets of ONE (sector, time slice) group ----
// The start hits are listed group by group (links.cuh: cells in (sector, slice, row) order); cell_offset is the exclusive
// scan of the per-cell start-hit counts and *total their sum.  One CTA; deterministic order.
__global__ void __launch_bounds__(kScanThreads) k_follow_chunk_list(const uint32_t* __restrict__ cell_offset, const uint32_t* __restrict__ total,
                                                                    int n_groups, int cells_per_group, uint2* __restrict__ chunks,
                                                                    int32_t* __restrict__ counters) {
  const uint32_t n_tl = (uint32_t)counters[kCntTracklets];
  uint32_t carry = 0;
  for (int base = 0; base < n_groups; base += kScanThreads) {
    const int g = base + (int)threadIdx.x;
    uint32_t lo = 0, hi = 0;
    if (g < n_groups) {
      lo = min(cell_offset[(size_t)g * cells_per_group], n_tl);
      hi = min(g + 1 < n_groups ? cell_offset[(size_t)(g + 1) * cells_per_group] : *total, n_tl);
    }
    const uint32_t nch = (hi - lo + kFrChunk - 1) / kFrChunk;
    uint32_t tot;
    uint32_t pos = carry + block_exclusive_scan(nch, tot);
    for (uint32_t k = 0; k < nch; ++k) chunks[pos + k] = make_uint2(lo + k * kFrChunk, min((uint32_t)kFrChunk, hi - lo - k * kFrChunk));
    carry += tot;
  }
  if (threadIdx.x == 0) counters[kCntChunks] = (int32_t)carry;
}

template <bool kDown>
__global__ void __launch_bounds__(kFrThreads, TPC_FR_MIN_CTAS) k_follow_rows(
    const float2* __restrict__ yt, const uint32_t* __restrict__ orig, const uint32_t* __restrict__ bin_start,
    TrackletSeeds seeds, int32_t* __restrict__ counters, const uint2* __restrict__ chunks, TrackletStore out,
    const __grid_constant__ Consts c) {
  extern __shared__ __align__(128) unsigned char fr_smem_raw[];
  FrSmem& sm = *reinterpret_cast<FrSmem*>(fr_smem_raw);
  const int tid = threadIdx.x;
  const unsigned lane = lane_id();
  const bool producer = tid == kFrWorkers;             // lane 0 of the extra warp requests the bulk copies
  for (int i = tid; i < c.n_rows; i += kFrThreads) { sm.xr[i] = c.xr[i]; sm.yoff[i] = c.yoff[i]; sm.pscale[i] = c.pscale[i]; }
  if (tid == 0) {
    for (int i = 0; i < kFrBinStages; ++i) mbar_init(&sm.bar_bins[i], 1);
    for (int i = 0; i < kFrHitStages; ++i) mbar_init(&sm.bar_hits[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const int n_chunks = counters[kCntChunks];
  uint32_t* queue = reinterpret_cast<uint32_t*>(counters + (kDown ? kCntQueueD : kCntQueueB));
  uint32_t n_steps = 0, n_upd = 0, n_cand = 0;
  const int last_row = kDown ? 0 : c.n_rows - 1;
  // widest window of a search + slack for the linear prediction, in grid time bins (a hint: a miss costs a global search)
  const int pad_gb = (int)(((c.win_slope * (__ldg(c.xr + 1) - __ldg(c.xr)) * (float)(c.miss_limit + 1) + c.win_const) * c.inv_Z + 2.0f) * c.inv_bin_w) + 1;
  const int cap_gb = (kFrBinsCap - 4) / c.n_pb;
  // Steps are numbered over the whole life of the CTA: step g uses offsets stage g % 4 and hits stage g % 3, and every
  // step index completes exactly one phase of each of its two barriers (parity = use count & 1).
  uint32_t itg0 = 0;

  for (;;) {
    __syncthreads();                                   // previous chunk fully retired (row tables / barriers visible)
    if (tid == 0) {
      sm.chunk = (int)atomicAdd(queue, 1u);
      sm.n_list[0] = sm.n_list[1] = sm.n_list[2] = 0;
      sm.acc_lo[0] = sm.acc_lo[1] = 0x7fffffff; sm.acc_hi[0] = sm.acc_hi[1] = -1;
      sm.r_first = kDown ? -1 : 0x7fffffff; sm.r_last_join = kDown ? 0x7fffffff : -1;
    }
    for (int i = tid; i < kFrJoinRows; i += kFrThreads) { sm.join_lo[i] = 0x7fffffff; sm.join_hi[i] = -1; }
    for (int i = tid; i < kRowStride + 2; i += kFrThreads) sm.join_cnt[i] = 0;
    __syncthreads();
    if (sm.chunk >= n_chunks) break;
    const uint2 ch = chunks[sm.chunk];
    const size_t j0 = ch.x;
    const int cnt = (int)ch.y;
    const int sr0 = seeds.a[j0].z;
    const int sr_base = sr0 - sr0 % c.n_rows;          // every tracklet of a chunk is in this sector

    // ---- prologue: states into shared memory, first target rows, the ranges the joining tracklets will need ----
    for (int slot = tid; slot < cnt; slot += kFrThreads) {
      const size_t j = j0 + slot;
      const int4 m = out.meta[j];
      const float4* rec = out.rec + 4 * j;
      const float4 q0 = rec[0], q1 = rec[1], q2 = rec[2], q3 = rec[3];      // (x, y, z, s) (t, k, c0, c1) (c2..c5) (d0, d1, d2, tstart)
      const int flags = m.x & ~kMetaHitsMask, n_hits = m.x & kMetaHitsMask;
      const int r_state = kDown ? m.y : m.z;           // row the state sits on: top of the chain (up) / first row (down)
      const bool active = kDown ? (!(flags & kMetaSkipFollowDown) && r_state > 0) : (!(flags & kMetaSkipFollowUp) && r_state < c.n_rows - 1);
      const int first = kDown ? r_state - 1 : r_state + 1;
      sm.first_row[slot] = active ? (uint8_t)first : (uint8_t)255;
      sm.r_init[slot] = (uint8_t)r_state;
      sm.packed[slot] = 0u | ((uint32_t)r_state << 8) | ((uint32_t)n_hits << 16) | ((uint32_t)r_state << 24);
      sm.state[0][slot] = q0; sm.state[1][slot] = q1; sm.state[2][slot] = q2; sm.state[3][slot] = q3;
      if (active) {
        if (kDown) { atomicMax(&sm.r_first, first); atomicMin(&sm.r_last_join, first); }
        else { atomicMin(&sm.r_first, first); atomicMax(&sm.r_last_join, first); }
        atomicAdd(&sm.join_cnt[first], 1);
        const float dxr = sm.xr[first] - sm.xr[r_state];
        const float dz_row = q1.x * dxr * rsqrtf(fmaxf(1.0f - q0.w * q0.w, 0.0025f));
#pragma unroll
        for (int k = 0; k < 3; ++k) {                  // the three rows it needs before its own steps feed the accumulators
          const int row = kDown ? first - k : first + k;
          if (row < 0 || row >= c.n_rows) break;
          const int gb = time_bin(q3.w + (q0.z + (float)(k + 1) * dz_row) * c.inv_Z, c);
          atomicMin(&sm.join_lo[row + 4], max(gb - pad_gb, 0));
          atomicMax(&sm.join_hi[row + 4], min(gb + pad_gb, c.n_tb - 1));
        }
      } else {                                         // nothing to follow: results = inputs (flags stripped from the hit count)
        if (!kDown) {
          out.cur[2 * j] = q0;
          out.cur[2 * j + 1] = make_float4(q1.x, q1.y, 0.0f, 0.0f);
        }
        reinterpret_cast<int*>(out.meta + j)[0] = n_hits;
      }
    }
    __syncthreads();
    const int r_first = sm.r_first, r_last_join = sm.r_last_join;
    if (kDown ? r_first < 0 : r_first >= c.n_rows) continue;       // no active tracklet in this chunk
    const int last_join_step = kDown ? r_first - r_last_join : r_last_join - r_first;
    if (tid < 32) {                                    // exclusive scan of the per-row join counts (one warp, 5 or 6 rows per lane)
      constexpr int kPer = (kRowStride + 2 + 31) / 32;
      int v[kPer], run = 0;
#pragma unroll
      for (int k = 0; k < kPer; ++k) { const int r = tid * kPer + k; v[k] = r < kRowStride + 2 ? sm.join_cnt[r] : 0; run += v[k]; }
      int inc = run;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, d); if ((int)lane >= d) inc += t; }
      int ex = inc - run;
#pragma unroll
      for (int k = 0; k < kPer; ++k) { const int r = tid * kPer + k; if (r < kRowStride + 2) { sm.join_off[r] = ex; sm.join_cnt[r] = ex; } ex += v[k]; }
    }
    __syncthreads();
    for (int slot = tid; slot < cnt; slot += kFrThreads) {
      const int fr = sm.first_row[slot];
      if (fr != 255) sm.join_sorted[atomicAdd(&sm.join_cnt[fr], 1)] = (uint16_t)slot;      // join_cnt doubles as the fill cursor
    }

    auto row_of = [&](int st) { return kDown ? r_first - st : r_first + st; };
    auto bin_stage = [&](int st) { return (int)((itg0 + (uint32_t)st) % kFrBinStages); };
    auto bin_parity = [&](int st) { return ((itg0 + (uint32_t)st) / kFrBinStages) & 1u; };
    auto hit_stage = [&](int st) { return (int)((itg0 + (uint32_t)st) % kFrHitStages); };
    auto hit_parity = [&](int st) { return ((itg0 + (uint32_t)st) / kFrHitStages) & 1u; };
    // producer side: grid offsets of step `st` (range = what the survivors predicted + the joiners' table), hits of step `st`
    auto issue_bins = [&](int st, int lo, int hi) {
      const int b = bin_stage(st);
      const int row = row_of(st);
      if (row >= 0 && row < c.n_rows) { lo = min(lo, sm.join_lo[row + 4]); hi = max(hi, sm.join_hi[row + 4]); }
      if (row < 0 || row >= c.n_rows || lo > hi) {
        sm.bst[b] = FrBinStage{0, 0, 0, 0};
        mbar_arrive(&sm.bar_bins[b]);
        return;
      }
      const int ngb = min(hi - lo + 1, cap_gb);
      const uint32_t b0 = grid_bin(sr_base + row, lo, 0, c);
      const uint32_t a0 = b0 & ~3u;
      const uint32_t n_copy = ((b0 - a0) + (uint32_t)(ngb * c.n_pb) + 1u + 3u) & ~3u;
      sm.bst[b] = FrBinStage{lo, ngb, (int)(b0 - a0), 0};
      mbar_arrive_expect_tx(&sm.bar_bins[b], n_copy * 4u);
      bulk_copy_g2s(sm.bins[b], bin_start + a0, n_copy * 4u, &sm.bar_bins[b]);
    };
    auto issue_hits = [&](int st) {
      const int b = bin_stage(st), h = hit_stage(st);
      mbar_wait(&sm.bar_bins[b], bin_parity(st));
      const FrBinStage bs = sm.bst[b];
      uint32_t lo = 0, n = 0;
      if (bs.ngb > 0) {
        const uint32_t h_lo = sm.bins[b][bs.off], h_hi = sm.bins[b][bs.off + bs.ngb * c.n_pb];
        lo = h_lo & ~1u;
        n = min(((h_hi - lo) + 1u) & ~1u, (uint32_t)kFrHitsCap);
      }
      sm.hst[h] = FrHitStage{lo, n};
      if (n > 0) {
        mbar_arrive_expect_tx(&sm.bar_hits[h], n * 8u);
        bulk_copy_g2s(sm.hits[h], yt + lo, n * 8u, &sm.bar_hits[h]);
      } else {
        mbar_arrive(&sm.bar_hits[h]);
      }
    };
    if (producer) {
      issue_bins(0, 0x7fffffff, -1); issue_bins(1, 0x7fffffff, -1); issue_bins(2, 0x7fffffff, -1);
      issue_hits(0); issue_hits(1);
    }
    __syncthreads();                                   // join_sorted complete

    // ---- the sweep ----
    int it = 0;
    for (;; ++it) {
      const int cur = it & 1, nxt = cur ^ 1;
      int* n_next = &sm.n_list[(it + 1) % 3];
      if (tid < kFrWorkers) {
        const int rt = row_of(it);                     // target row of this step
        const int n_surv = sm.n_list[it % 3];
        const int j_off = sm.join_off[rt], n_act = n_surv + (sm.join_off[rt + 1] - j_off);
        const int bst_i = bin_stage(it), hst_i = hit_stage(it);
        mbar_wait(&sm.bar_bins[bst_i], bin_parity(it));
        mbar_wait(&sm.bar_hits[hst_i], hit_parity(it));
        const FrBinStage bs = sm.bst[bst_i];
        const FrHitStage hs = sm.hst[hst_i];
        const uint32_t* s_bins = sm.bins[bst_i] + bs.off;
        const float2* s_hits = sm.hits[hst_i];
        const float xn = sm.xr[rt];
        const float yoff_r = sm.yoff[rt], pscale_r = sm.pscale[rt];
        int* row_hit_rt = out.row_hit + (j0 * kRowStride + rt);
        int w_lo = 0x7fffffff, w_hi = -1;              // this thread's share of the predicted range of step it + 3

        for (int base = (tid & ~31); base < n_act; base += kFrWorkers) {
          const int i = base + (int)lane;
          const bool valid = i < n_act;
          int slot = 0;
          if (valid) slot = i < n_surv ? (int)sm.list[cur][i] : (int)sm.join_sorted[j_off + (i - n_surv)];
          bool keep = false;
          if (valid) {
            TrackState S;
            float tstart;
            {
              const float4 q0 = sm.state[0][slot], q1 = sm.state[1][slot], q2 = sm.state[2][slot], q3 = sm.state[3][slot];
              S.x = q0.x; S.y = q0.y; S.z = q0.z; S.s = q0.w; S.t = q1.x; S.k = q1.y; S.c0 = q1.z; S.c1 = q1.w;
              S.c2 = q2.x; S.c3 = q2.y; S.c4 = q2.z; S.c5 = q2.w; S.d0 = q3.x; S.d1 = q3.y; S.d2 = q3.z; tstart = q3.w;
            }
            uint32_t packed = sm.packed[slot];
            const float z_old = S.z;
            const bool ok = transport(S, xn, c.cB, c.sin_phi_max);
            ++n_steps;
            bool end_dir = !ok;
            if (ok) {
              const int r_last = (int)((packed >> 8) & 255u);
              const float w = c.win_slope * fabsf(xn - sm.xr[r_last]) + c.win_const;
              // ---- window search in the staged row ----
              const float tpred = tstart + S.z * c.inv_Z;
              const float hw = w * c.inv_Z + 0.05f;    // superset margins; the exact predicate decides
              const float yw = w + 0.01f;
              const int tb_lo = time_bin(tpred - hw, c), tb_hi = time_bin(tpred + hw, c);
              const int pb0 = pad_bin(S.y - yw, yoff_r, pscale_r, c), pb1 = pad_bin(S.y + yw, yoff_r, pscale_r, c);
              bool fast = tb_lo >= bs.gb0 && tb_hi < bs.gb0 + bs.ngb && tb_hi <= tb_lo + 1;
              uint32_t lo0 = 0, n0 = 0, lo1 = 0, n_all = 0;
              if (fast) {
                const uint32_t* sb = s_bins + (tb_lo - bs.gb0) * c.n_pb + pb0;
                const int np = pb1 - pb0 + 1;
                lo0 = sb[0];
                uint32_t hi_all = sb[np];
                n0 = hi_all - lo0; n_all = n0;
                if (tb_hi != tb_lo) { lo1 = sb[c.n_pb]; hi_all = sb[c.n_pb + np]; n_all += hi_all - lo1; }
                fast = lo0 >= hs.lo && hi_all <= hs.lo + hs.n;
              }
              int m = -1;
              float hy = 0.0f, ht = 0.0f;              // the attached hit
              if (fast) {
                float bdd = __int_as_float(0x7f800000);
                bool tie = false;
                n_cand += n_all;
                lo0 -= hs.lo; lo1 -= hs.lo + n0;       // candidate i lives at s_hits[(i < n0 ? lo0 : lo1) + i]
#pragma unroll 1
                for (uint32_t i2 = 0; i2 < n_all; ++i2) {
                  const uint32_t q = (i2 < n0 ? lo0 : lo1) + i2;
                  const float2 cq = s_hits[q];
                  const float ey = cq.x - S.y;
                  const float ez = (cq.y - tstart) * c.Z - S.z;
                  const float dd = ey * ey + ez * ez;
                  const bool in = fabsf(ey) < w && fabsf(ez) < w;
                  tie = tie || (in && dd == bdd);
                  if (in && dd < bdd) { bdd = dd; m = (int)q; hy = cq.x; ht = cq.y; }
                }
                if (tie) fast = false;                 // rare (exact fp32 tie): decided on the original index, in global memory
                else if (m >= 0) m += (int)hs.lo;
              }
              if (!fast) {
                count_rare(counters, 3);
                m = search_row_global(yt, orig, bin_start, sr_base + rt, S.y, S.z, tstart, w, yoff_r, pscale_r, c, counters);
                if (m >= 0) { const float2 hit = yt[m]; hy = hit.x; ht = hit.y; }
              }
              row_hit_rt[(size_t)slot * kRowStride] = m;
              if (m >= 0) {
                kalman_update(S, hy, (ht - tstart) * c.Z, c.ry, c.rz);
                ++n_upd;
                packed = (packed & 0x00ff0000u) + 0x00010000u + ((uint32_t)rt << 8) + ((uint32_t)rt << 24);      // misses = 0, r_last = r_ext = rt, ++hits
              } else {
                if ((packed & 255u) == 0u && (packed >> 24) != (uint32_t)sm.r_init[slot]) {
                  // first miss after an update: the state BEFORE this transport -- still in shared memory -- is the state
                  // after the last update
                  float4* rec = out.rec + 4 * (j0 + slot);
                  rec[0] = lds128_volatile(&sm.state[0][slot]); rec[1] = lds128_volatile(&sm.state[1][slot]);
                  rec[2] = lds128_volatile(&sm.state[2][slot]); rec[3] = lds128_volatile(&sm.state[3][slot]);
                }
                ++packed;
                if ((int)(packed & 255u) == c.miss_limit) end_dir = true;
              }
              if (rt == last_row) end_dir = true;
              if (!end_dir) {
                sm.state[0][slot] = make_float4(S.x, S.y, S.z, S.s);
                sm.state[1][slot] = make_float4(S.t, S.k, S.c0, S.c1);
                sm.state[2][slot] = make_float4(S.c2, S.c3, S.c4, S.c5);
                sm.state[3][slot] = make_float4(S.d0, S.d1, S.d2, tstart);
                sm.packed[slot] = packed;
                keep = true;
                // where it will look three rows on (prefetch hint): z moves on by what it moved in this step
                const int gb = time_bin(tstart + (S.z + 3.0f * (S.z - z_old)) * c.inv_Z, c);
                w_lo = min(w_lo, gb); w_hi = max(w_hi, gb);
              }
            }
            if (end_dir) {                             // the direction ends here: S = state after the last transport
              const size_t j = j0 + slot;
              if ((packed & 255u) == 0u && (packed >> 24) != (uint32_t)sm.r_init[slot]) store_rec(out.rec + 4 * j, S, tstart);   // ... = state after the last update
              if (!kDown) {
                out.cur[2 * j] = make_float4(S.x, S.y, S.z, S.s);
                out.cur[2 * j + 1] = make_float4(S.t, S.k, 0.0f, 0.0f);
              }
              int* mp = reinterpret_cast<int*>(out.meta + j);
              mp[0] = (int)((packed >> 16) & 255u);
              mp[kDown ? 1 : 2] = (int)(packed >> 24);
            }
          }
          // survivors onto the next step's list
          const unsigned mk = __ballot_sync(0xffffffffu, keep);
          if (mk) {
            int pos = 0;
            const int leader = __ffs(mk) - 1;
            if ((int)lane == leader) pos = atomicAdd(n_next, __popc(mk));
            pos = __shfl_sync(0xffffffffu, pos, leader);
            if (keep) sm.list[nxt][pos + __popc(mk & ((1u << lane) - 1u))] = (uint16_t)slot;
          }
        }
        // the warp's predicted range into the accumulator of step it + 3
        w_lo = __reduce_min_sync(0xffffffffu, w_lo); w_hi = __reduce_max_sync(0xffffffffu, w_hi);
        if (lane == 0 && w_lo <= w_hi) { atomicMin(&sm.acc_lo[cur], w_lo); atomicMax(&sm.acc_hi[cur], w_hi); }
      } else if (producer) {
        sm.n_list[(it + 2) % 3] = 0;                   // the list length this step neither reads nor appends to
      }
      __syncthreads();
      if (*n_next == 0 && it + 1 > last_join_step) break;
      if (producer) {
        int lo = sm.acc_lo[cur], hi = sm.acc_hi[cur];
        sm.acc_lo[cur] = 0x7fffffff; sm.acc_hi[cur] = -1;
        if (lo <= hi) { lo = max(lo - pad_gb, 0); hi = min(hi + pad_gb, c.n_tb - 1); }
        issue_bins(it + 3, lo, hi);
        issue_hits(it + 2);
      }
    }
    // drain the copies requested for steps that will not run: offsets of it + 1, it + 2, hits of it + 1 (and complete the
    // phase of the one hits stage that was never requested), so that the next chunk starts at step it + 3
    if (producer) {
      mbar_wait(&sm.bar_bins[bin_stage(it + 1)], bin_parity(it + 1));
      mbar_wait(&sm.bar_bins[bin_stage(it + 2)], bin_parity(it + 2));
      mbar_wait(&sm.bar_hits[hit_stage(it + 1)], hit_parity(it + 1));
      mbar_arrive(&sm.bar_hits[hit_stage(it + 2)]);
    }
    itg0 += (uint32_t)it + 3u;
  }
  add_work_counters(counters, kDown ? 3 : 1, n_steps, n_upd, n_cand);
}

}  // namespace tpc
