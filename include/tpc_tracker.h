/* tpc_tracker.h -- C-ABI boundary of the B200-native TPC time-frame tracker.
 *
 * What it is: the step the paper names as "the most computing-intense workload of the synchronous
 * reconstruction" (§1): TPC sector tracking of a whole continuous-readout time frame held in
 * GPU memory -- cellular-automaton seeding in native (pad row, pad, time) coordinates ("the track seeding
 * operates using the time as coordinate instead of the spatial z coordinate") followed by
 * Kalman-filter track following, "derived from the Run 2 HLT TPC tracking", with "the
 * reusage of memory for sequential steps of the tracking algorithm".
 * The entry points and their argument lists are fixed by BASELINE.json L5 (north_star):
 *   tpc_tracker_create(geometry, params), tpc_track_timeframe(clusters, n, stream, tracks_out),
 *   tpc_tracker_destroy.  The exact operations (steps C1..C6) are defined in DESIGN.md §3.
 * After the hot path, three widening steps are separate calls on the tracker's outputs:
 *   tpc_merge_tracks (C7), tpc_refit_chains (C8), tpc_vertex_time (C9), ... tpc_refit_full (C12); DESIGN.md §3 defines them too.
 *
 * Conventions
 *   - Plain C, no torch types.  Every pointer is marked DEVICE or HOST.
 *   - Return value: 0 (TPC_OK) or a negative tpc_status_t.  tpc_strerror() names it.
 *   - Ownership: the CALLER owns cluster arrays, output arrays and the scratch arena; the handle owns only
 *     small geometry tables (a few KB of device memory) and CUDA events.  Inputs are never written.
 *   - tpc_track_timeframe only enqueues work on `cuda_stream`: it never synchronises and never allocates.
 *     One call in flight per handle; a handle is not thread-safe.
 *   - All kernels are hand-written CUDA for sm_100a.  There is no CPU fallback: without a CUDA device
 *     tpc_tracker_create fails with TPC_ECUDA.
 */
#ifndef TPC_TRACKER_H_
#define TPC_TRACKER_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tpc_tracker tpc_tracker_t; /* opaque */

typedef enum {
  TPC_OK = 0,
  TPC_EINVAL = -1, /* null pointer, bad geometry / params, n < 0, n > max_clusters, n >= 2^31           */
  TPC_ENOMEM = -2, /* arena missing or smaller than tpc_tracker_arena_bytes()                            */
  TPC_ECUDA = -3   /* a CUDA runtime call or kernel launch failed (also: no CUDA device)                 */
} tpc_status_t;

/* Bits of the device status word tpc_tracks_t::status (0 = everything fitted). */
enum {
  TPC_STATUS_TRACKLET_OVERFLOW = 1,  /* more start hits than max_tracklets: the excess was dropped       */
  TPC_STATUS_TRACK_OVERFLOW = 2,     /* more tracks than max_tracks: *n_tracks holds the required count  */
  TPC_STATUS_TRACK_HIT_OVERFLOW = 4, /* more track hits than max_track_hits                              */
  TPC_STATUS_INVALID_CLUSTERS = 8    /* some clusters lay outside the geometry and were ignored          */
};

/* One parametric geometry serves all configs (BASELINE.json L7, L8).  Sector s of a 36-sector TPC is
 * s < 18: A side, s >= 18: C side; every sector is tracked in its own local frame.                       */
typedef struct {
  int32_t n_sectors;     /* 1 or 36                                                                     */
  int32_t n_rows;        /* 152 (3 <= n_rows <= 160)                                                    */
  float x0_cm;           /* 85.0   x_r = (float)((double)x0_cm + (double)row_pitch_cm * r)              */
  float row_pitch_cm;    /* 1.07                                                                        */
  float pad_pitch_cm;    /* 0.5                                                                         */
  float tan_half_sector; /* (float)tan(10 deg); pads_r = floor(2 x_r tan / pad_pitch) in double         */
  float time_bin_cm;     /* 0.516 = 2.58 cm/us * 0.2 us                                                 */
  float drift_len_cm;    /* 250 (informative)                                                           */
  float max_time_bin;    /* upper bound of the time coordinate in a frame; sizes the grid; < 2^19 bins
                            (the grid lookups' absolute fp32 margins hold up to there), else TPC_EINVAL */
} tpc_geometry_t;

typedef struct {
  float win_slope, win_const;     /* 0.05, 0.5 : window W(dx) = win_slope*|dx| + win_const [cm] (BASELINE L7) */
  float chi2_cut;                 /* 9 : mid-point deviation chi2 of a hit triplet            (BASELINE L7) */
  int32_t miss_limit, min_hits;   /* 10, 30                                                   (BASELINE L7) */
  float sigma_y_cm, sigma_z_cm;   /* hit errors used by the tracker (reading A4)                  */
  float slope_y_max, slope_z_max; /* 1.0, 1.5 : neighbour search area half size per cm of dx  (reading A1)  */
  int32_t seed_min_hits;          /* 3 : reciprocal chain length that makes a start hit       (reading A7)  */
  float sin_phi_max;              /* 0.95                                                     (reading A12) */
  float inv_R_per_qpt;            /* (float)(1/666.7) : curvature [1/cm] per q/pT [1/GeV]     (BASELINE L7) */
  float c0_y2, c0_s2, c0_k2, c0_z2, c0_t2; /* initial / reset covariance diagonal             (reading A8)  */
  int32_t grid_time_bins;         /* width of one grid bin in time bins; 0 = default: 8, or 9 / 10 when that makes
                                     the grid bin index -- the radix sort key -- one digit size shorter          */
  int32_t grid_pad_bins;          /* grid bins across a pad row; 0 = default (8); lowered automatically so that
                                     no lookup window spans more than two of them.  The grid only accelerates:
                                     results do not depend on either value.                                  */
  int32_t slice_time_bins;        /* tracklets are constructed in (sector, time slice, row) order for cache
                                     locality; width of a slice in time bins; 0 = default (256)              */
  int32_t follower;               /* 0 = one lane per tracklet, persistent warps with lane refill, lookups in global
                                     memory (csrc/tracklet.cuh); 1 = row-synchronous: a CTA sweeps the pad rows in lock
                                     step with the row's grid offsets and hits staged in shared memory by bulk copies
                                     (csrc/follow_rows.cuh; measured slower; kept for A/B).  Same results. */
  int64_t max_clusters;           /* capacity: largest n of any tpc_track_timeframe call                    */
  int64_t max_tracklets;          /* capacity of the tracklet store; 0 = max_clusters/10 + 4096             */
  int64_t max_tracks;             /* host entry point only: staging capacity; 0 = max_clusters/64 + 4096    */
  int64_t max_track_hits;         /* host entry point only: staging capacity; 0 = max_clusters              */
  void* arena;                    /* DEVICE, caller-owned scratch (e.g. a torch uint8 tensor), 256-B aligned */
  size_t arena_bytes;
  int32_t host_staging;           /* 1: reserve arena space for tpc_track_timeframe_host                    */
  int32_t profile;                /* 1: record a CUDA event after every step (tpc_tracker_step_ms)          */
} tpc_params_t;

/* fp32 SoA clusters, n entries each.  row[i] = sector*n_rows + pad_row as an integer-valued float (exact
 * below 2^24); pad in pad units (pad p covers [p-0.5, p+0.5)); time in time bins; charge is never read.   */
typedef struct {
  const float* row;
  const float* pad;
  const float* time;
  const float* charge; /* may be NULL */
} tpc_clusters_t;

/* Caller-allocated output buffers and their capacities.  DEVICE pointers for tpc_track_timeframe, HOST
 * pointers for tpc_track_timeframe_host.  Track order is by ascending internal tracklet slot and is
 * deterministic; `seed_hit` (original index of the start hit) is the unique key of a track.               */
typedef struct {
  int32_t max_tracks;
  int64_t max_track_hits;
  int32_t* n_tracks;     /* scalar: number of tracks found (may exceed max_tracks, see status)              */
  int64_t* n_track_hits; /* scalar                                                                          */
  int32_t* status;       /* scalar: TPC_STATUS_* bits                                                       */
  int32_t *seed_hit, *sector, *first_row, *last_row, *n_hits; /* [max_tracks]                               */
  int64_t* hit_offset;   /* [max_tracks] first entry of the track in hit_index                              */
  float *x, *y, *z_rel, *time_ref, *sin_phi, *dzds, *q_pt;    /* [max_tracks] state after the tracklet's last Kalman
                            update: at its innermost hit, unless the downward refit FAILed early (about 1 track in
                            1000: the state then sits on a higher pad row -- x says which).  z_rel [cm] is relative
                            to time_ref [time bins] (reading A2)                                      */
  float* cov9;           /* [max_tracks*9] (yy, ys, ss, yk, sk, kk | zz, zt, tt); may be NULL               */
  int32_t* hit_index;    /* [max_track_hits] original cluster indices, ascending row, per track contiguous  */
  /* parity taps, each may be NULL (device entry point only): */
  int32_t *link_up, *link_down;   /* [n] indexed AND valued by original cluster index, -1 = none, after cleaning */
  uint8_t* is_start_hit;          /* [n] by original index                                                  */
  int32_t max_tracklets;          /* capacity of the four tracklet taps                                     */
  int32_t* n_tracklets;           /* scalar: number of tracklets (= start hits) constructed                 */
  int32_t* tracklet_seed;         /* [max_tracklets] original index of the start hit                        */
  int32_t* tracklet_n_hits;       /* [max_tracklets]                                                        */
  int32_t* tracklet_row_hit;      /* [max_tracklets*n_rows] original indices, -1 = none                     */
  float* tracklet_par;            /* [max_tracklets*7] (x, y, z_rel, sin_phi, dzds, q_pt, time_ref)         */
  /* optional, each may be NULL (device entry point only; tpc_refit_chains needs both): the coordinates of the track
   * hits, so that a later pass over a track's hits reads them in order instead of gathering from the clusters       */
  float* hit_y_time;              /* [max_track_hits*2] (y [cm] = (pad - c_r) * pad_pitch, time [bins]) of hit_index[k] */
  uint8_t* hit_row;               /* [max_track_hits] pad row of hit_index[k]                                */
} tpc_tracks_t;

/* Bytes of arena the tracker needs for params->max_clusters (the `max_clusters` argument, if > 0,
 * overrides it).  Host-side arithmetic only; needs no device.  Returns 0 on invalid arguments.            */
size_t tpc_tracker_arena_bytes(const tpc_geometry_t* geometry, const tpc_params_t* params, int64_t max_clusters);

/* Validates, builds the per-row tables in double (rounded once to fp32), uploads them and plans the arena
 * (lifetime-based reuse across steps).  Errors: TPC_EINVAL, TPC_ENOMEM, TPC_ECUDA.          */
int tpc_tracker_create(const tpc_geometry_t* geometry, const tpc_params_t* params, tpc_tracker_t** out);

/* Tracks one time frame: steps C1 ingest -> C2 neighbours finder -> C3/C4 cleaner + start hits ->
 * C5 tracklet constructor -> C6 selector, all enqueued on `cuda_stream` (a cudaStream_t; NULL = default).
 * `clusters` holds DEVICE pointers.  Asynchronous.  Device-detected overflow sets *status.                  */
int tpc_track_timeframe(tpc_tracker_t* tracker, const tpc_clusters_t* clusters, int64_t n, void* cuda_stream,
                        tpc_tracks_t* tracks_out);

/* Same, with HOST buffers (pinned for full speed): copies row/pad/time host->device into arena staging,
 * tracks, copies the scalars and exactly the produced tracks / hits back, and synchronises the stream
 * before returning.  Needs params->host_staging = 1 at create time.  Taps are ignored.                     */
int tpc_track_timeframe_host(tpc_tracker_t* tracker, const tpc_clusters_t* host_clusters, int64_t n,
                             void* cuda_stream, tpc_tracks_t* host_tracks_out);

/* With params->profile = 1: milliseconds of each step of the last completed call (synchronises on the
 * handle's last event).  ms_out[0..n_steps) in the order of tpc_tracker_step_name().  Returns the number of
 * steps, or a negative status.                                                                              */
int tpc_tracker_step_ms(tpc_tracker_t* tracker, float* ms_out, int32_t capacity);
const char* tpc_tracker_step_name(int32_t step);

/* Number of kernel launches the last tpc_track_timeframe call enqueued (memsets not counted).              */
int64_t tpc_tracker_last_launches(const tpc_tracker_t* tracker);

/* Work counters of the last completed tpc_track_timeframe call, read back from the device (synchronises
 * `cuda_stream`).  The block lives in memory the handle owns, not in the arena, so it stays valid after
 * tpc_merge_tracks / tpc_refit_chains (which reuse the arena):
 * out[0] tracklets constructed, [1] start hits found, [2] invalid clusters, [3] row steps (transports) of the
 * tracklet constructor, [4] Kalman updates, [5] candidates scanned by its window searches (each the sum over the
 * four phase kernels), then [6 + 3 p + k] the same three counts (k = 0 row steps, 1 updates, 2 candidates) of phase
 * p = 0 chain fit, 1 follow up, 2 refit down, 3 follow down.  These are the units of the constructor's roofline
 * (DESIGN.md §6).  Then the rare paths taken: [18] refits replayed after a failed transport that followed a hole,
 * [19] refits that failed before their first update (the up pass's state is the result), [20] window searches that met
 * an exact fp32 tie of the smallest distance (decided on the original index), [21] window searches of the row-synchronous
 * follower that were served from global memory because the staged range did not cover them.  Returns the number of
 * counters (22) or a negative status.                                                                                                 */
int tpc_tracker_work_counters(tpc_tracker_t* tracker, void* cuda_stream, int64_t* out, int32_t capacity);

/* Arena plan: for allocation i writes name, offset, bytes, first and last step of its lifetime.
 * Returns the number of allocations; i out of range returns -1.                                            */
int tpc_tracker_arena_plan(const tpc_tracker_t* tracker, int32_t i, const char** name, size_t* offset,
                           size_t* bytes, int32_t* first_step, int32_t* last_step);

/* Self test of the constructor's arithmetic (synchronises `cuda_stream`; allocates 16 bytes for its duration): the
 * range-restricted square root and reciprocal sequences used by the Kalman transport / update are compared with the
 * IEEE-754 correctly rounded sqrtf(x) and 1.0f / x over EVERY fp32 bit pattern of their ranges.  mismatches_out
 * (HOST, 2 entries) receives the number of differing bit patterns for sqrt and for the reciprocal (both must be 0:
 * the decision arithmetic has to round like the definition, BASELINE.json L5).                              */
int tpc_selftest_fast_math(void* cuda_stream, uint64_t* mismatches_out);

/* Micro-benchmark of the bound the tracklet constructor is accounted against ("measure it with a
 * micro-benchmark, do not quote a datasheet number"): dependency-free streams of fp32 multiplies and adds -- no FMA
 * contraction, like the constructor's arithmetic (--fmad=false) -- on every SM, timed with CUDA events on
 * `cuda_stream` (synchronises it).  lane_inst_per_s_out (HOST, 2 entries): [0] scalar FMUL / FADD instructions,
 * in lane-instructions per second (warp instructions x 32) -- the "alu" peak of the roofline; [1] the same arithmetic
 * issued as packed mul.f32x2 / add.f32x2 (two fp32 operations per lane-instruction), in fp32 operations per second.
 * Returns TPC_OK or TPC_ECUDA.                                                                              */
int tpc_selftest_alu_peak(void* cuda_stream, double* lane_inst_per_s_out);

/* ---- C0: the TPC cluster finder, the step in front of the path (clusterization is part
 * of the synchronous GPU load; DESIGN.md §3 "C0", readings D1..D6).  Zero-suppressed ADC samples in, clusters in the tracker's
 * input format out: a sample is a peak iff adc >= peak_threshold and it beats its (up to) 8 neighbours in (pad, time) of the
 * same sector-row (larger adc; ties to the earlier sample); a peak's cluster is the fp32 centre of gravity of its 3 x 3 window. */
typedef struct {
  const int32_t* row;    /* DEVICE [n_digits] sector * n_rows + pad row                                                  */
  const int32_t* pad;    /* DEVICE [n_digits] pad                                                                        */
  const int32_t* time;   /* DEVICE [n_digits] time bin.  Samples are sorted by (row, time, pad), no duplicates (reading D1:
                            the readout order); an unsorted input gives unspecified clusters, never an out-of-bounds access */
  const float* adc;      /* DEVICE [n_digits] ADC count                                                                  */
} tpc_digits_t;

typedef struct { float peak_threshold; /* 8 : smallest ADC of a cluster's peak sample (reading D4) */ } tpc_cluster_params_t;

typedef struct {   /* caller-allocated DEVICE buffers: exactly the arrays tpc_clusters_t takes                              */
  int64_t max_clusters;
  float *row, *pad, *time, *charge;   /* [max_clusters], in the input order of the peak samples                          */
  int64_t* n_clusters;   /* scalar: clusters found (may exceed max_clusters: the first max_clusters are written)         */
  int32_t* status;       /* scalar: 1 = more clusters than max_clusters                                                  */
} tpc_clusters_out_t;

/* Arena bytes the call needs for n_digits samples (host arithmetic, 16 B per sample: the staged clusters; 0 = invalid).   */
size_t tpc_cluster_finder_scratch_bytes(int64_t n_digits);

/* Asynchronous on `cuda_stream`, never allocates: scratch = the handle's arena (the call precedes tpc_track_timeframe on the
 * same stream, which then overwrites it).  Errors: TPC_EINVAL, TPC_ENOMEM (arena smaller than the scratch), TPC_ECUDA.
 * tpc_merge_last_launches() reports its launches.                                                                       */
int tpc_find_clusters(tpc_tracker_t* tracker, const tpc_cluster_params_t* params, const tpc_digits_t* digits, int64_t n_digits,
                      void* cuda_stream, tpc_clusters_out_t* clusters_out);

/* ---- C0 for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same cluster finder, needing NO tracker handle and NO arena.  Its scratch (16 B per sample) is a fixed
 * array inside the library image, so every GPU that loads the library holds 16.1 MiB for it until the process exits, and one
 * call handles at most tpc_find_clusters_static_max_digits() = 1 048 576 samples (larger n: TPC_ENOMEM, nothing enqueued --
 * use tpc_find_clusters).  Arguments, results (bit-identical to tpc_find_clusters) and the other errors as there.  The call
 * enqueues one memset and five kernels on `cuda_stream` and calls no cudaMalloc / cudaFree or allocating routine.
 * ALL calls on one GPU share the one scratch array: calls that overlap on the GPU (different streams without ordering, or
 * different host threads) race -- order them on one stream or with events.
 * tpc_find_clusters_static_setup() looks the array's device address up for the CURRENT device (once per device; also done by
 * the first call on a device): call it before a stream capture begins.  Errors: TPC_ECUDA.                                 */
int64_t tpc_find_clusters_static_max_digits(void);
int tpc_find_clusters_static_setup(void);
int tpc_find_clusters_static(const tpc_cluster_params_t* params, const tpc_digits_t* digits, int64_t n_digits,
                             void* cuda_stream, tpc_clusters_out_t* clusters_out);

/* ---- C7: sector-boundary merging of the per-sector tracks (DESIGN.md §3 "C7", readings M1..M8; PAPER.md L23 / L25:
 * "full TPC tracking" -- the sector tracker is followed by a merger of the sector tracks; BASELINE.json L8: 36 sectors,
 * each in its rotated local frame).  A widening step after the hot path (linking only: the
 * refit of a merged chain and central-electrode crossings are not part of it).                                  */
typedef struct {
  float cut_y_cm, cut_z_cm;         /* 2, 2     : |dy|, |dz| between the extrapolated inner piece and the outer piece   */
  float cut_sin_phi, cut_q_pt;      /* 0.05, 0.5: |d sin phi|, |d q/pT| [c/GeV]                            (reading M4) */
  int32_t max_row_gap;              /* 12 : the outer piece's state row r_B <= last_row_A + 1 + max_row_gap (reading M5);
                                       always r_B > max(first_row_A, state row of A) and r_B <= first_row_B (M7)        */
  int32_t max_row_overlap;          /* 2  : r_B >= last_row_A + 1 - max_row_overlap                                     */
} tpc_merge_params_t;

/* Caller-allocated DEVICE buffers, [tracks->max_tracks] each (entries >= *n_tracks are -1).                       */
typedef struct {
  int32_t* next;     /* track index of the outer continuation of track i, -1 = none                               */
  int32_t* prev;     /* track index of the inner piece that track i continues, -1 = none                          */
  int32_t* root;     /* first piece of i's chain (i itself for an unmerged track)                                  */
  int32_t* n_links;  /* scalar: number of links (merged tracks = *n_tracks - *n_links)                             */
} tpc_merged_t;

/* Bytes of the tracker's arena that tpc_merge_tracks uses for `max_tracks` tracks (host arithmetic; 0 = invalid).  */
size_t tpc_merge_scratch_bytes(const tpc_tracker_t* tracker, int64_t max_tracks);

/* Links the tracks that `tracks` (DEVICE buffers, as written by tpc_track_timeframe of THIS tracker: geometry, row
 * table and curvature constant are the handle's) holds across sector boundaries of the same TPC side.  Asynchronous on
 * `cuda_stream`; reads *tracks->n_tracks on the device; never allocates: its scratch is the handle's arena, whose
 * tracking scratch is dead once tpc_track_timeframe has been enqueued on the same stream (the two calls must not
 * overlap on different streams).  The result does not depend on the order of the tracks.
 * Errors: TPC_EINVAL (null pointer, non-positive cut), TPC_ENOMEM (arena smaller than tpc_merge_scratch_bytes),
 * TPC_ECUDA.                                                                                                     */
int tpc_merge_tracks(tpc_tracker_t* tracker, const tpc_merge_params_t* merge_params, const tpc_tracks_t* tracks,
                     void* cuda_stream, tpc_merged_t* merged_out);

/* ---- C10: merging across the CENTRAL ELECTRODE (DESIGN.md §3 "C10", readings CE1..CE6; PAPER.md L23:
 * the z of a hit is only known through its time).  A track that approaches the electrode (dz/ds > 0 in the time-derived
 * coordinate) continues in the mirror sector (S + 18) mod 36 of the other TPC side: x, y, sin phi, q/pT continuous, the time
 * coordinate reflected.  Row window and reciprocal best match as in C7; needs the 36-sector geometry (else nothing links). */
typedef struct {
  float cut_y_cm, cut_z_cm;         /* 2, 2     : |dy|; distance of the crossing from the gap between the two pieces [cm]    */
  float cut_sin_phi, cut_q_pt;      /* 0.05, 0.5                                                                             */
  float cut_dzds;                   /* 0.1      : |dz/ds of A + dz/ds of B| (mirrored slopes)                   (reading CE5) */
  int32_t max_row_gap, max_row_overlap;   /* 12, 2 : as in tpc_merge_params_t                                                 */
} tpc_ce_params_t;

typedef struct {   /* caller-allocated DEVICE buffers, [tracks->max_tracks] each                                               */
  int32_t* next;     /* the continuation of track i behind the electrode, -1 = none                                          */
  int32_t* prev;     /* the piece in front of the electrode that track i continues, -1 = none                                */
  float* t_ce;       /* time coordinate [time bins] at which linked track i crosses the electrode = (t0 v_drift + drift
                        length) / time bin: the collision time, with no vertex assumption; 0 for unlinked tracks             */
  int32_t* n_links;  /* scalar                                                                                               */
} tpc_ce_merged_t;

/* Same calling rules as tpc_merge_tracks (asynchronous, scratch = the handle's arena, tpc_merge_scratch_bytes of it, after
 * tpc_track_timeframe on the same stream; it may follow tpc_merge_tracks, whose scratch it overwrites).  Errors: TPC_EINVAL,
 * TPC_ENOMEM, TPC_ECUDA.  tpc_merge_last_launches() then reports this call's launches.                                       */
int tpc_merge_central_electrode(tpc_tracker_t* tracker, const tpc_ce_params_t* ce_params, const tpc_tracks_t* tracks,
                                void* cuda_stream, tpc_ce_merged_t* merged_out);

/* ---- C8: refit of the chains linked by C7 (DESIGN.md §3 "C8", readings F1..F6): one inward Kalman pass over the hits
 * all pieces of a chain own, each piece in its own sector frame, state and covariance rotated at every boundary.      */
typedef struct {   /* caller-allocated DEVICE buffers, indexed by track like tpc_tracks_t                              */
  int32_t* ok;           /* [max_tracks] 1: root of a chain of >= 2 pieces, refitted; 0: anything else (values passed
                            through); -1: root whose refit failed (a transport / rotation reached sin_phi_max, or a
                            hit list of the chain was cut by TPC_STATUS_TRACK_HIT_OVERFLOW)                            */
  int32_t* chain_hits;   /* [max_tracks] hits of the whole chain (roots), else the track's own n_hits                  */
  int32_t* chain_pieces; /* [max_tracks] pieces of the chain (roots), else 1                                           */
  float* par7;           /* [max_tracks*7] (x, y, z_rel, sin_phi, dzds, q_pt, time_ref) at the innermost hit of the root */
  float* cov9;           /* [max_tracks*9] (yy, ys, ss, yk, sk, kk | zz, zt, tt); zeros unless ok == 1                  */
} tpc_refit_t;

/* `tracks` are the outputs of tpc_track_timeframe INCLUDING the optional hit_y_time / hit_row arrays (the hits'
 * coordinates are read from them, in order), `merged` those of tpc_merge_tracks; all on the same stream, after
 * tpc_merge_tracks.  Asynchronous; never allocates (4 bytes of arena per track).  Errors: TPC_EINVAL (also: hit
 * coordinates missing), TPC_ENOMEM, TPC_ECUDA.  tpc_merge_last_launches() then reports this call's launches.          */
int tpc_refit_chains(tpc_tracker_t* tracker, const tpc_tracks_t* tracks, const tpc_merged_t* merged, void* cuda_stream,
                     tpc_refit_t* refit_out);

/* ---- C11: track-based hit rejection and track-model residual coding, the step behind the path (
 * "removal of TPC hits of tracks not used for physics, reduction of the hit property entropy"; DESIGN.md §3
 * "C11", readings R11-1..R11-6).  The entropy coder that would follow (ANS) is out of scope.                                 */
typedef struct {
  float reject_q_pt;     /* 1/0.15 : hits owned by a track with |q/pT| above this are rejected                  (R11-1) */
  float step_y_cm;       /* 0.025  : quantisation step of the residual in y                                      (R11-3) */
  float step_z_cm;       /* 0.025  : ... in the time-derived coordinate z = time * time_bin_cm                           */
} tpc_compress_params_t;

typedef struct {   /* caller-allocated DEVICE buffers                                                                    */
  uint8_t* reject;   /* [n_clusters] by ORIGINAL cluster index: 1 = the hit belongs to a rejected track                  */
  int32_t* ok;       /* [max_tracks] 1: coded; -1: rejected; 0: not coded (a transport reached sin_phi_max, or the hit
                        list was cut by TPC_STATUS_TRACK_HIT_OVERFLOW): its symbols are 0 from the failing hit on         */
  int16_t* res_y;    /* [max_track_hits] symbol of hit_index[k]: rintf((y - predicted y) / step_y), clamped to +-32767    */
  int16_t* res_z;    /* [max_track_hits] ... of (time - time_ref) * time_bin_cm against the predicted z                  */
} tpc_compressed_t;

/* `tracks` = the outputs of tpc_track_timeframe INCLUDING cov9 and the optional hit_y_time / hit_row arrays.  A track's
 * header (its seven parameters, cov9, n_hits, the hit rows) plus its symbols reproduce every hit to within half a step: the
 * prediction is a Kalman filter started from the header and updated with the reconstructed hits (closed loop).
 * Asynchronous on `cuda_stream`, after tpc_track_timeframe; uses 256 bytes of the arena.  Errors: TPC_EINVAL, TPC_ENOMEM,
 * TPC_ECUDA.  tpc_merge_last_launches() reports its launches.                                                             */
int tpc_compress_tracks(tpc_tracker_t* tracker, const tpc_compress_params_t* params, const tpc_tracks_t* tracks,
                        int64_t n_clusters, void* cuda_stream, tpc_compressed_t* out);

/* ---- C12: refit with the full 5x5 covariance, multiple scattering and energy loss (§2:
 * the planned "improvement of the tracking efficiency, which will require the fit of more tracks and more attached hits";
 * DESIGN.md §3 "C12", readings FF1..FF7).  One inward Kalman pass over the hits of every ROOT of the chains of tpc_merge_tracks,
 * single tracks included: state (y, z, sin_phi, dzds, q_pt) at x, the full symmetric covariance, process noise of multiple
 * scattering (Highland's theta0 without the logarithm) and the mean energy loss dE/dx = dedx_mip / beta^2 of the drift gas.   */
typedef struct {
  float inv_x0_per_cm;        /* 1 / radiation length of the gas, e.g. 1 / 3e4; >= 0                                          */
  float dedx_mip_gev_per_cm;  /* stopping power of a minimum-ionising particle, e.g. 1.7e-6; >= 0                             */
  float mass_gev;             /* mass hypothesis, e.g. 0.13957 (pion); >= 0                                                   */
  float eloss_sigma;          /* relative width of the energy loss (straggling), e.g. 0.1; >= 0                               */
} tpc_fullfit_params_t;

typedef struct {   /* caller-allocated DEVICE buffers, indexed by track like tpc_tracks_t                                     */
  int32_t* ok;           /* [max_tracks] 1: root, refitted; 0: not a root (values passed through); -1: root whose refit failed
                            (a transport / rotation reached sin_phi_max, or a hit list was cut by TPC_STATUS_TRACK_HIT_OVERFLOW) */
  int32_t* chain_hits;   /* [max_tracks] hits of the whole chain (roots), else the track's own n_hits                         */
  int32_t* chain_pieces; /* [max_tracks] pieces of the chain (roots), else 1                                                  */
  float* par7;           /* [max_tracks*7] (x, y, z_rel, sin_phi, dzds, q_pt, time_ref) at the innermost hit of the root;
                            the track's own parameters unless ok == 1                                                         */
  float* cov15;          /* [max_tracks*15] lower triangle in the order (y, z, sin_phi, dzds, q_pt):
                            yy | zy zz | sy sz ss | ty tz ts tt | ky kz ks kt kk; zeros unless ok == 1                        */
} tpc_fullfit_t;

/* Same calling rules as tpc_refit_chains (`tracks` with hit_y_time / hit_row, `merged` from tpc_merge_tracks, same stream,
 * asynchronous, 512 + 4 bytes of arena per track).  Errors: TPC_EINVAL (null pointer, negative parameter, hit coordinates
 * missing), TPC_ENOMEM, TPC_ECUDA.  tpc_merge_last_launches() then reports this call's launches.                             */
int tpc_refit_full(tpc_tracker_t* tracker, const tpc_fullfit_params_t* params, const tpc_tracks_t* tracks,
                   const tpc_merged_t* merged, void* cuda_stream, tpc_fullfit_t* out);

/* The same refit over chains that may CONTINUE BEHIND THE CENTRAL ELECTRODE (DESIGN.md §3 reading FF8): `ce_merged` = the output
 * of tpc_merge_central_electrode for the same tracks (NULL = tpc_refit_full).  The link e -> b of C10 is used where e has no
 * sector-boundary continuation and b continues nothing across a sector boundary; b is then no root (ok = 0, values passed
 * through) and the root of e's chain is fitted over the hits of both sides: at the electrode the time coordinate is reflected
 * about t_ce[e] (z = (2 t_ce - time_ref_b - time_ref_e) time_bin_cm - z, dzds = -dzds, covariance D P D), x, y, sin_phi, q_pt
 * are continuous.  Same calling rules and errors as tpc_refit_full; the links must be C10's (reciprocal).                     */
int tpc_refit_full_ce(tpc_tracker_t* tracker, const tpc_fullfit_params_t* params, const tpc_tracks_t* tracks,
                      const tpc_merged_t* merged, const tpc_ce_merged_t* ce_merged, void* cuda_stream, tpc_fullfit_t* out);

/* ---- C9: where and when a track passes the beam line (DESIGN.md §3 "C9"; z is only known once the
 * collision time is).  Every state of `par7` (DEVICE, [max_tracks*7] = (x, y, z_rel, sin_phi, dzds, q_pt, time_ref): the
 * par7 of tpc_refit_chains, or the same seven values of tpc_tracks_t) is transported to x = 0, the beam axis in every
 * sector frame: vertex_time = time_ref + z / time_bin_cm [time bins] = (t0 v_drift + drift_len - side z_vertex) / time_bin_cm
 * for a primary track, vertex_y [cm] its offset from the axis; ok = 0 (outputs 0) when sin phi would reach sin_phi_max.
 * Outputs: DEVICE, [max_tracks].  Asynchronous, reads *n_tracks on the device.  Errors: TPC_EINVAL, TPC_ECUDA.          */
int tpc_vertex_time(tpc_tracker_t* tracker, const int32_t* n_tracks, int32_t max_tracks, const float* par7,
                    void* cuda_stream, int32_t* ok, float* vertex_time, float* vertex_y);

/* Number of kernel launches the last tpc_merge_tracks call enqueued (memsets not counted).                        */
int64_t tpc_merge_last_launches(const tpc_tracker_t* tracker);

int tpc_tracker_destroy(tpc_tracker_t* tracker);

const char* tpc_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* TPC_TRACKER_H_ */
