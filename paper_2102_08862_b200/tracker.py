"""Thin Python binding of the C-ABI in ``include/tpc_tracker.h`` (same names; argument marshalling only).

PyTorch is used for device memory and streams, nothing else: every step of the path runs in the CUDA kernels of
``csrc/``.  There is no CPU fallback -- a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from dataclasses import dataclass

from . import build as _build

TPC_OK, TPC_EINVAL, TPC_ENOMEM, TPC_ECUDA = 0, -1, -2, -3
STATUS_TRACKLET_OVERFLOW, STATUS_TRACK_OVERFLOW, STATUS_TRACK_HIT_OVERFLOW, STATUS_INVALID_CLUSTERS = 1, 2, 4, 8

EXPORTS = ("tpc_tracker_arena_bytes", "tpc_tracker_create", "tpc_track_timeframe", "tpc_track_timeframe_host",
           "tpc_tracker_step_ms", "tpc_tracker_step_name", "tpc_tracker_last_launches", "tpc_tracker_work_counters",
           "tpc_tracker_arena_plan", "tpc_selftest_fast_math", "tpc_selftest_alu_peak",
           "tpc_cluster_finder_scratch_bytes", "tpc_find_clusters",
           "tpc_find_clusters_static_max_digits", "tpc_find_clusters_static_setup", "tpc_find_clusters_static",
           "tpc_merge_scratch_bytes", "tpc_merge_tracks", "tpc_merge_central_electrode", "tpc_refit_chains", "tpc_refit_full", "tpc_refit_full_ce", "tpc_vertex_time", "tpc_compress_tracks", "tpc_merge_last_launches",
           "tpc_tracker_destroy", "tpc_strerror")


class Geometry(C.Structure):
    """``tpc_geometry_t``"""
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("x0_cm", C.c_float), ("row_pitch_cm", C.c_float),
                ("pad_pitch_cm", C.c_float), ("tan_half_sector", C.c_float), ("time_bin_cm", C.c_float),
                ("drift_len_cm", C.c_float), ("max_time_bin", C.c_float)]


class Params(C.Structure):
    """``tpc_params_t``"""
    _fields_ = [("win_slope", C.c_float), ("win_const", C.c_float), ("chi2_cut", C.c_float),
                ("miss_limit", C.c_int32), ("min_hits", C.c_int32), ("sigma_y_cm", C.c_float), ("sigma_z_cm", C.c_float),
                ("slope_y_max", C.c_float), ("slope_z_max", C.c_float), ("seed_min_hits", C.c_int32),
                ("sin_phi_max", C.c_float), ("inv_R_per_qpt", C.c_float),
                ("c0_y2", C.c_float), ("c0_s2", C.c_float), ("c0_k2", C.c_float), ("c0_z2", C.c_float), ("c0_t2", C.c_float),
                ("grid_time_bins", C.c_int32), ("grid_pad_bins", C.c_int32), ("slice_time_bins", C.c_int32), ("follower", C.c_int32),
                ("max_clusters", C.c_int64), ("max_tracklets", C.c_int64),
                ("max_tracks", C.c_int64), ("max_track_hits", C.c_int64), ("arena", C.c_void_p), ("arena_bytes", C.c_size_t),
                ("host_staging", C.c_int32), ("profile", C.c_int32)]


class Clusters(C.Structure):
    """``tpc_clusters_t``"""
    _fields_ = [("row", C.c_void_p), ("pad", C.c_void_p), ("time", C.c_void_p), ("charge", C.c_void_p)]


class Tracks(C.Structure):
    """``tpc_tracks_t``"""
    _fields_ = [("max_tracks", C.c_int32), ("max_track_hits", C.c_int64),
                ("n_tracks", C.c_void_p), ("n_track_hits", C.c_void_p), ("status", C.c_void_p),
                ("seed_hit", C.c_void_p), ("sector", C.c_void_p), ("first_row", C.c_void_p), ("last_row", C.c_void_p),
                ("n_hits", C.c_void_p), ("hit_offset", C.c_void_p),
                ("x", C.c_void_p), ("y", C.c_void_p), ("z_rel", C.c_void_p), ("time_ref", C.c_void_p),
                ("sin_phi", C.c_void_p), ("dzds", C.c_void_p), ("q_pt", C.c_void_p), ("cov9", C.c_void_p),
                ("hit_index", C.c_void_p), ("link_up", C.c_void_p), ("link_down", C.c_void_p), ("is_start_hit", C.c_void_p),
                ("max_tracklets", C.c_int32), ("n_tracklets", C.c_void_p), ("tracklet_seed", C.c_void_p),
                ("tracklet_n_hits", C.c_void_p), ("tracklet_row_hit", C.c_void_p), ("tracklet_par", C.c_void_p),
                ("hit_y_time", C.c_void_p), ("hit_row", C.c_void_p)]


class MergeParams(C.Structure):
    """``tpc_merge_params_t``"""
    _fields_ = [("cut_y_cm", C.c_float), ("cut_z_cm", C.c_float), ("cut_sin_phi", C.c_float), ("cut_q_pt", C.c_float),
                ("max_row_gap", C.c_int32), ("max_row_overlap", C.c_int32)]


class Merged(C.Structure):
    """``tpc_merged_t``"""
    _fields_ = [("next", C.c_void_p), ("prev", C.c_void_p), ("root", C.c_void_p), ("n_links", C.c_void_p)]


class Digits(C.Structure):
    """``tpc_digits_t``"""
    _fields_ = [("row", C.c_void_p), ("pad", C.c_void_p), ("time", C.c_void_p), ("adc", C.c_void_p)]


class ClusterParams(C.Structure):
    """``tpc_cluster_params_t``"""
    _fields_ = [("peak_threshold", C.c_float)]


class ClustersOut(C.Structure):
    """``tpc_clusters_out_t``"""
    _fields_ = [("max_clusters", C.c_int64), ("row", C.c_void_p), ("pad", C.c_void_p), ("time", C.c_void_p), ("charge", C.c_void_p),
                ("n_clusters", C.c_void_p), ("status", C.c_void_p)]


class CompressParams(C.Structure):
    """``tpc_compress_params_t``"""
    _fields_ = [("reject_q_pt", C.c_float), ("step_y_cm", C.c_float), ("step_z_cm", C.c_float)]


class Compressed(C.Structure):
    """``tpc_compressed_t``"""
    _fields_ = [("reject", C.c_void_p), ("ok", C.c_void_p), ("res_y", C.c_void_p), ("res_z", C.c_void_p)]


class CeParams(C.Structure):
    """``tpc_ce_params_t``"""
    _fields_ = [("cut_y_cm", C.c_float), ("cut_z_cm", C.c_float), ("cut_sin_phi", C.c_float), ("cut_q_pt", C.c_float),
                ("cut_dzds", C.c_float), ("max_row_gap", C.c_int32), ("max_row_overlap", C.c_int32)]


class CeMerged(C.Structure):
    """``tpc_ce_merged_t``"""
    _fields_ = [("next", C.c_void_p), ("prev", C.c_void_p), ("t_ce", C.c_void_p), ("n_links", C.c_void_p)]


def default_ce_params() -> CeParams:
    """DESIGN.md §3 C10 reading CE5."""
    return CeParams(2.0, 2.0, 0.05, 0.5, 0.1, 12, 2)


class Refit(C.Structure):
    """``tpc_refit_t``"""
    _fields_ = [("ok", C.c_void_p), ("chain_hits", C.c_void_p), ("chain_pieces", C.c_void_p), ("par7", C.c_void_p), ("cov9", C.c_void_p)]


class FullFitParams(C.Structure):
    """``tpc_fullfit_params_t``"""
    _fields_ = [("inv_x0_per_cm", C.c_float), ("dedx_mip_gev_per_cm", C.c_float), ("mass_gev", C.c_float), ("eloss_sigma", C.c_float)]


class FullFit(C.Structure):
    """``tpc_fullfit_t``"""
    _fields_ = [("ok", C.c_void_p), ("chain_hits", C.c_void_p), ("chain_pieces", C.c_void_p), ("par7", C.c_void_p), ("cov15", C.c_void_p)]


DEFAULT_FULLFIT_PARAMS = (1.0 / 3.0e4, 1.7e-6, 0.13957, 0.1)      # DESIGN.md §3 C12 reading FF3: the drift gas, pions


def default_merge_params() -> MergeParams:
    """DESIGN.md §3 C7 readings M4 / M5."""
    return MergeParams(2.0, 2.0, 0.05, 0.5, 12, 2)


def default_geometry(n_sectors: int = 36, max_time_bin: float = 487.0) -> Geometry:
    """BASELINE.json L7: 152 rows at 85.0 + 1.07 r cm, 0.5 cm pads, +-10 degree sectors, 0.516 cm time bins."""
    return Geometry(n_sectors, 152, 85.0, 1.07, 0.5, math.tan(math.radians(10.0)), 0.516, 250.0, max_time_bin)


def default_params(sigma_y: float = 0.08, sigma_z: float = 0.12, max_clusters: int = 0) -> Params:
    """BASELINE.json L7 cuts and the readings of DESIGN.md §3."""
    return Params(win_slope=0.05, win_const=0.5, chi2_cut=9.0, miss_limit=10, min_hits=30,
                  sigma_y_cm=sigma_y, sigma_z_cm=sigma_z, slope_y_max=1.0, slope_z_max=1.5, seed_min_hits=3,
                  sin_phi_max=0.95, inv_R_per_qpt=1.0 / 666.7, c0_y2=1.0, c0_s2=0.1, c0_k2=100.0, c0_z2=1.0, c0_t2=0.1,
                  grid_time_bins=0, grid_pad_bins=0, slice_time_bins=0, follower=0, max_clusters=max_clusters, max_tracklets=0, max_tracks=0, max_track_hits=0,
                  arena=None, arena_bytes=0, host_staging=0, profile=0)


_lib = None


def load_library(build_if_missing: bool = True):
    """Loads ``csrc/libtpctracker.so`` (building it in-tree if missing or stale).  Raises if that fails."""
    global _lib
    if _lib is None:
        path = _build.build_cuda() if build_if_missing else _build.LIB
        if not os.path.exists(path):
            raise RuntimeError(f"CUDA library {path} is missing; run __graft_entry__.build()")
        L = C.CDLL(path)
        vp = C.c_void_p
        L.tpc_tracker_arena_bytes.argtypes = [C.POINTER(Geometry), C.POINTER(Params), C.c_int64]
        L.tpc_tracker_arena_bytes.restype = C.c_size_t
        L.tpc_tracker_create.argtypes = [C.POINTER(Geometry), C.POINTER(Params), C.POINTER(vp)]
        L.tpc_track_timeframe.argtypes = [vp, C.POINTER(Clusters), C.c_int64, vp, C.POINTER(Tracks)]
        L.tpc_track_timeframe_host.argtypes = [vp, C.POINTER(Clusters), C.c_int64, vp, C.POINTER(Tracks)]
        L.tpc_tracker_step_ms.argtypes = [vp, C.POINTER(C.c_float), C.c_int32]
        L.tpc_tracker_step_name.argtypes = [C.c_int32]
        L.tpc_tracker_step_name.restype = C.c_char_p
        L.tpc_tracker_last_launches.argtypes = [vp]
        L.tpc_tracker_last_launches.restype = C.c_int64
        L.tpc_tracker_work_counters.argtypes = [vp, vp, C.POINTER(C.c_int64), C.c_int32]
        L.tpc_tracker_arena_plan.argtypes = [vp, C.c_int32, C.POINTER(C.c_char_p), C.POINTER(C.c_size_t),
                                             C.POINTER(C.c_size_t), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        L.tpc_tracker_destroy.argtypes = [vp]
        L.tpc_selftest_fast_math.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.tpc_selftest_fast_math.restype = C.c_int
        L.tpc_selftest_alu_peak.argtypes = [vp, C.POINTER(C.c_double)]
        L.tpc_selftest_alu_peak.restype = C.c_int
        L.tpc_merge_scratch_bytes.argtypes = [vp, C.c_int64]
        L.tpc_merge_scratch_bytes.restype = C.c_size_t
        L.tpc_merge_tracks.argtypes = [vp, C.POINTER(MergeParams), C.POINTER(Tracks), vp, C.POINTER(Merged)]
        L.tpc_merge_tracks.restype = C.c_int
        L.tpc_cluster_finder_scratch_bytes.argtypes = [C.c_int64]
        L.tpc_cluster_finder_scratch_bytes.restype = C.c_size_t
        L.tpc_find_clusters.argtypes = [vp, C.POINTER(ClusterParams), C.POINTER(Digits), C.c_int64, vp, C.POINTER(ClustersOut)]
        L.tpc_find_clusters.restype = C.c_int
        L.tpc_find_clusters_static_max_digits.argtypes = []
        L.tpc_find_clusters_static_max_digits.restype = C.c_int64
        L.tpc_find_clusters_static_setup.argtypes = []
        L.tpc_find_clusters_static_setup.restype = C.c_int
        L.tpc_find_clusters_static.argtypes = [C.POINTER(ClusterParams), C.POINTER(Digits), C.c_int64, vp, C.POINTER(ClustersOut)]
        L.tpc_find_clusters_static.restype = C.c_int
        L.tpc_merge_central_electrode.argtypes = [vp, C.POINTER(CeParams), C.POINTER(Tracks), vp, C.POINTER(CeMerged)]
        L.tpc_merge_central_electrode.restype = C.c_int
        L.tpc_refit_chains.argtypes = [vp, C.POINTER(Tracks), C.POINTER(Merged), vp, C.POINTER(Refit)]
        L.tpc_refit_chains.restype = C.c_int
        L.tpc_refit_full.argtypes = [vp, C.POINTER(FullFitParams), C.POINTER(Tracks), C.POINTER(Merged), vp, C.POINTER(FullFit)]
        L.tpc_refit_full.restype = C.c_int
        L.tpc_refit_full_ce.argtypes = [vp, C.POINTER(FullFitParams), C.POINTER(Tracks), C.POINTER(Merged), C.POINTER(CeMerged), vp, C.POINTER(FullFit)]
        L.tpc_refit_full_ce.restype = C.c_int
        L.tpc_compress_tracks.argtypes = [vp, C.POINTER(CompressParams), C.POINTER(Tracks), C.c_int64, vp, C.POINTER(Compressed)]
        L.tpc_compress_tracks.restype = C.c_int
        L.tpc_vertex_time.argtypes = [vp, vp, C.c_int32, vp, vp, vp, vp, vp]
        L.tpc_vertex_time.restype = C.c_int
        L.tpc_merge_last_launches.argtypes = [vp]
        L.tpc_merge_last_launches.restype = C.c_int64
        L.tpc_strerror.argtypes = [C.c_int]
        L.tpc_strerror.restype = C.c_char_p
        for nm in ("tpc_tracker_create", "tpc_track_timeframe", "tpc_track_timeframe_host", "tpc_tracker_step_ms",
                   "tpc_tracker_work_counters", "tpc_tracker_arena_plan", "tpc_tracker_destroy"):
            getattr(L, nm).restype = C.c_int
        _lib = L
    return _lib


class TpcError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {load_library().tpc_strerror(code).decode()} ({code})")


def tpc_selftest_fast_math(stream=None) -> tuple:
    """(sqrt mismatches, reciprocal mismatches) of the constructor's range-restricted sqrt / reciprocal against the
    IEEE results over every fp32 bit pattern of their ranges (include/tpc_tracker.h); both must be 0."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("tpc_selftest_fast_math needs a CUDA device")
    s = stream if stream is not None else torch.cuda.current_stream()
    out = (C.c_uint64 * 2)()
    rc = load_library().tpc_selftest_fast_math(C.c_void_p(s.cuda_stream), out)
    if rc != TPC_OK:
        raise TpcError(rc, "tpc_selftest_fast_math")
    return int(out[0]), int(out[1])


def tpc_find_clusters_static_max_digits() -> int:
    """Largest n one ``tpc_find_clusters_static`` call accepts."""
    return int(load_library().tpc_find_clusters_static_max_digits())


def tpc_find_clusters_static_setup() -> None:
    """Looks up the built-in scratch array of the CURRENT device (once per device; call before a stream capture)."""
    rc = load_library().tpc_find_clusters_static_setup()
    if rc != TPC_OK:
        raise TpcError(rc, "tpc_find_clusters_static_setup")


def tpc_find_clusters_static(row, pad, time, adc, out, n: int | None = None, peak_threshold: float = 8.0, stream=None):
    """C0 without a tracker handle, an arena or any allocation (include/tpc_tracker.h): DEVICE int32 (row, pad, time) / float32
    adc in, the caller's ``out`` = (row, pad, time, charge float32[max_clusters], n_clusters int64[1], status int32[1]) DEVICE
    tensors filled.  Argument marshalling only: nothing is allocated here either."""
    import torch
    n = int(adc.shape[0]) if n is None else int(n)
    for t_, dt in ((row, torch.int32), (pad, torch.int32), (time, torch.int32), (adc, torch.float32)):
        if not (t_.is_cuda and t_.dtype == dt and t_.is_contiguous() and t_.shape[0] >= n):
            raise ValueError("digits must be contiguous CUDA tensors: int32 row / pad / time, float32 adc, length >= n")
    K = int(out[0].shape[0])
    dg = Digits(row.data_ptr(), pad.data_ptr(), time.data_ptr(), adc.data_ptr())
    co = ClustersOut(K, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), out[3].data_ptr(), out[4].data_ptr(), out[5].data_ptr())
    cp = ClusterParams(float(peak_threshold))
    s = stream if stream is not None else torch.cuda.current_stream(adc.device)
    rc = load_library().tpc_find_clusters_static(C.byref(cp), C.byref(dg), n, C.c_void_p(s.cuda_stream), C.byref(co))
    if rc != TPC_OK:
        raise TpcError(rc, "tpc_find_clusters_static")
    return out


def tpc_selftest_alu_peak(stream=None) -> tuple:
    """(scalar fp32 multiply / add lane-instructions per second, fp32 operations per second issued as packed f32x2)
    measured by the library's micro-benchmark (include/tpc_tracker.h): the "alu" peak of the constructor's roofline."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("tpc_selftest_alu_peak needs a CUDA device")
    s = stream if stream is not None else torch.cuda.current_stream()
    out = (C.c_double * 2)()
    rc = load_library().tpc_selftest_alu_peak(C.c_void_p(s.cuda_stream), out)
    if rc != TPC_OK:
        raise TpcError(rc, "tpc_selftest_alu_peak")
    return float(out[0]), float(out[1])


def tpc_tracker_arena_bytes(geometry: Geometry, params: Params, max_clusters: int = 0) -> int:
    return int(load_library().tpc_tracker_arena_bytes(C.byref(geometry), C.byref(params), int(max_clusters)))


@dataclass
class TrackResult:
    """Device (or pinned host) tensors written by one call; ``n_tracks`` etc. are 0-dim-like 1-element tensors."""
    n_tracks: object
    n_track_hits: object
    status: object
    seed_hit: object
    sector: object
    first_row: object
    last_row: object
    n_hits: object
    hit_offset: object
    x: object
    y: object
    z_rel: object
    time_ref: object
    sin_phi: object
    dzds: object
    q_pt: object
    cov9: object
    hit_index: object
    link_up: object = None
    link_down: object = None
    is_start_hit: object = None
    n_tracklets: object = None
    tracklet_seed: object = None
    tracklet_n_hits: object = None
    tracklet_row_hit: object = None
    tracklet_par: object = None
    hit_y_time: object = None      # optional: (y, time) of every track hit, in hit_index order (needed by tpc_refit_chains)
    hit_row: object = None


class Tracker:
    """``tpc_tracker_create`` / ``tpc_track_timeframe`` / ``tpc_tracker_destroy`` with torch-owned buffers."""

    def __init__(self, geometry: Geometry, params: Params, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the tracker has no CPU fallback")
        self._torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        self.geometry = geometry
        self.params = Params.from_buffer_copy(params)
        need = self.lib.tpc_tracker_arena_bytes(C.byref(geometry), C.byref(self.params), 0)
        if need == 0:
            raise TpcError(TPC_EINVAL, "tpc_tracker_arena_bytes")
        with torch.cuda.device(self.device):
            self.arena = torch.empty(int(need) + 256, dtype=torch.uint8, device=self.device)
            base = (self.arena.data_ptr() + 255) // 256 * 256
            self.params.arena = base
            self.params.arena_bytes = int(need)
            self.handle = C.c_void_p()
            rc = self.lib.tpc_tracker_create(C.byref(geometry), C.byref(self.params), C.byref(self.handle))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_tracker_create")
        self.arena_bytes = int(need)

    # -- buffers ---------------------------------------------------------------------------------------------
    def _alloc_outputs(self, n: int, max_tracks: int, max_track_hits: int, taps: bool, max_tracklets: int, host: bool,
                       hit_coords: bool = False, tap_row_hit: bool = True):
        torch = self._torch
        kw = dict(device="cpu", pin_memory=True) if host else dict(device=self.device)
        e = lambda shape, dt: torch.empty(shape, dtype=dt, **kw)
        K, H = max_tracks, max_track_hits
        r = TrackResult(
            n_tracks=e(1, torch.int32), n_track_hits=e(1, torch.int64), status=e(1, torch.int32),
            seed_hit=e(K, torch.int32), sector=e(K, torch.int32), first_row=e(K, torch.int32), last_row=e(K, torch.int32),
            n_hits=e(K, torch.int32), hit_offset=e(K, torch.int64),
            x=e(K, torch.float32), y=e(K, torch.float32), z_rel=e(K, torch.float32), time_ref=e(K, torch.float32),
            sin_phi=e(K, torch.float32), dzds=e(K, torch.float32), q_pt=e(K, torch.float32), cov9=e((K, 9), torch.float32),
            hit_index=e(H, torch.int32))
        if taps:
            nr = self.geometry.n_rows
            r.link_up, r.link_down, r.is_start_hit = e(n, torch.int32), e(n, torch.int32), e(n, torch.uint8)
            r.n_tracklets = e(1, torch.int32)
            r.tracklet_seed, r.tracklet_n_hits = e(max_tracklets, torch.int32), e(max_tracklets, torch.int32)
            r.tracklet_row_hit = e((max_tracklets, nr), torch.int32) if tap_row_hit else None
            r.tracklet_par = e((max_tracklets, 7), torch.float32)
        if hit_coords and not host:
            r.hit_y_time, r.hit_row = e((H, 2), torch.float32), e(H, torch.uint8)
        return r

    @staticmethod
    def _tracks_struct(r: TrackResult, max_tracks: int, max_track_hits: int, max_tracklets: int) -> Tracks:
        p = lambda t: (t.data_ptr() if t is not None else None)
        return Tracks(max_tracks, max_track_hits, p(r.n_tracks), p(r.n_track_hits), p(r.status), p(r.seed_hit), p(r.sector),
                      p(r.first_row), p(r.last_row), p(r.n_hits), p(r.hit_offset), p(r.x), p(r.y), p(r.z_rel), p(r.time_ref),
                      p(r.sin_phi), p(r.dzds), p(r.q_pt), p(r.cov9), p(r.hit_index), p(r.link_up), p(r.link_down),
                      p(r.is_start_hit), max_tracklets, p(r.n_tracklets), p(r.tracklet_seed), p(r.tracklet_n_hits),
                      p(r.tracklet_row_hit), p(r.tracklet_par), p(r.hit_y_time), p(r.hit_row))

    def default_capacities(self, n: int):
        return max(n // 64 + 4096, 1), max(n, 1)

    def alloc_outputs(self, n: int, taps: bool = False, host: bool = False, max_tracks: int = 0, max_track_hits: int = 0,
                      hit_coords: bool = False, tap_row_hit: bool = True):
        K, H = self.default_capacities(n)
        K, H = (max_tracks or K), (max_track_hits or H)
        T = int(self.params.max_tracklets or (self.params.max_clusters // 10 + 4096)) if taps else 0
        out = self._alloc_outputs(n, K, H, taps, T, host, hit_coords, tap_row_hit)
        return out, self._tracks_struct(out, K, H, T)

    # -- the C-ABI calls -------------------------------------------------------------------------------------
    def tpc_track_timeframe(self, row, pad, time, n: int | None = None, outputs=None, taps: bool = False, stream=None):
        """Device tensors in, device tensors out; asynchronous on ``stream`` (default: torch's current stream)."""
        torch = self._torch
        n = int(row.shape[0]) if n is None else int(n)
        for t in (row, pad, time):
            if not (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.shape[0] >= n):
                raise ValueError("clusters must be contiguous float32 CUDA tensors of length >= n")
        if outputs is None:
            outputs = self.alloc_outputs(n, taps=taps)
        out, st = outputs
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        cl = Clusters(row.data_ptr(), pad.data_ptr(), time.data_ptr(), None)
        rc = self.lib.tpc_track_timeframe(self.handle, C.byref(cl), n, C.c_void_p(s.cuda_stream), C.byref(st))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_track_timeframe")
        return out

    def tpc_track_timeframe_host(self, row, pad, time, n: int | None = None, outputs=None, stream=None):
        """Host (pinned) tensors in and out; H2D + tracking + D2H inside the call; synchronous."""
        torch = self._torch
        n = int(row.shape[0]) if n is None else int(n)
        for t in (row, pad, time):
            if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
                raise ValueError("clusters must be contiguous float32 host tensors")
        if outputs is None:
            outputs = self.alloc_outputs(n, host=True, max_tracks=int(self.params.max_tracks or 0),
                                         max_track_hits=int(self.params.max_track_hits or 0))
        out, st = outputs
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        cl = Clusters(row.data_ptr(), pad.data_ptr(), time.data_ptr(), None)
        rc = self.lib.tpc_track_timeframe_host(self.handle, C.byref(cl), n, C.c_void_p(s.cuda_stream), C.byref(st))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_track_timeframe_host")
        return out

    def tpc_find_clusters(self, row, pad, time, adc, n: int | None = None, max_clusters: int | None = None, peak_threshold: float = 8.0,
                          out=None, stream=None):
        """C0 on DEVICE int32 (row, pad, time) / float32 adc tensors sorted by (row, time, pad); returns
        (row, pad, time, charge, n_clusters, status) device tensors -- the first three are ``tpc_track_timeframe``'s input."""
        torch = self._torch
        n = int(adc.shape[0]) if n is None else int(n)
        for t_, dt in ((row, torch.int32), (pad, torch.int32), (time, torch.int32), (adc, torch.float32)):
            if not (t_.is_cuda and t_.dtype == dt and t_.is_contiguous() and t_.shape[0] >= n):
                raise ValueError("digits must be contiguous CUDA tensors: int32 row / pad / time, float32 adc, length >= n")
        K = int(max_clusters) if max_clusters is not None else max(n, 1)
        if out is None:
            e = lambda dt, k=K: torch.empty(max(k, 1), dtype=dt, device=self.device)
            out = (e(torch.float32), e(torch.float32), e(torch.float32), e(torch.float32), e(torch.int64, 1), e(torch.int32, 1))
        dg = Digits(row.data_ptr(), pad.data_ptr(), time.data_ptr(), adc.data_ptr())
        co = ClustersOut(K, out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr(), out[3].data_ptr(), out[4].data_ptr(), out[5].data_ptr())
        cp = ClusterParams(float(peak_threshold))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self.lib.tpc_find_clusters(self.handle, C.byref(cp), C.byref(dg), n, C.c_void_p(s.cuda_stream), C.byref(co))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_find_clusters")
        return out

    def tpc_merge_tracks(self, outputs, merge_params: MergeParams | None = None, merged=None, stream=None):
        """C7 on the DEVICE outputs of ``tpc_track_timeframe`` (same stream); returns (next, prev, root, n_links) tensors."""
        torch = self._torch
        out, st = outputs
        K = int(st.max_tracks)
        if merged is None:
            merged = tuple(torch.empty(max(K, 1), dtype=torch.int32, device=self.device) for _ in range(3)) + \
                     (torch.empty(1, dtype=torch.int32, device=self.device),)
        mp = merge_params if merge_params is not None else default_merge_params()
        m = Merged(*(t.data_ptr() for t in merged))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self.lib.tpc_merge_tracks(self.handle, C.byref(mp), C.byref(st), C.c_void_p(s.cuda_stream), C.byref(m))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_merge_tracks")
        return merged

    def tpc_merge_central_electrode(self, outputs, ce_params: CeParams | None = None, merged=None, stream=None):
        """C10 on the DEVICE outputs of ``tpc_track_timeframe`` (same stream); returns (next, prev, t_ce, n_links) tensors."""
        torch = self._torch
        out, st = outputs
        K = max(int(st.max_tracks), 1)
        if merged is None:
            e = lambda dt: torch.empty(K, dtype=dt, device=self.device)
            merged = (e(torch.int32), e(torch.int32), e(torch.float32), torch.empty(1, dtype=torch.int32, device=self.device))
        mp = ce_params if ce_params is not None else default_ce_params()
        m = CeMerged(*(t.data_ptr() for t in merged))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self.lib.tpc_merge_central_electrode(self.handle, C.byref(mp), C.byref(st), C.c_void_p(s.cuda_stream), C.byref(m))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_merge_central_electrode")
        return merged

    def tpc_refit_chains(self, outputs, merged, refit=None, stream=None):
        """C8 on the DEVICE track outputs (allocated with ``hit_coords=True``) and C7 links (same stream); returns
        (ok, chain_hits, chain_pieces, par7, cov9)."""
        torch = self._torch
        out, st = outputs
        K = max(int(st.max_tracks), 1)
        if refit is None:
            e = lambda shape, dt: torch.empty(shape, dtype=dt, device=self.device)
            refit = (e(K, torch.int32), e(K, torch.int32), e(K, torch.int32), e((K, 7), torch.float32), e((K, 9), torch.float32))
        m = Merged(*(t.data_ptr() for t in merged))
        r = Refit(*(t.data_ptr() for t in refit))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self.lib.tpc_refit_chains(self.handle, C.byref(st), C.byref(m), C.c_void_p(s.cuda_stream), C.byref(r))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_refit_chains")
        return refit

    def tpc_refit_full(self, outputs, merged, full_params=DEFAULT_FULLFIT_PARAMS, out=None, stream=None, ce_merged=None):
        """C12 on the DEVICE track outputs (allocated with ``hit_coords=True``) and C7 links (same stream); with ``ce_merged``
        (the tensors of ``tpc_merge_central_electrode``) over chains that continue behind the central electrode
        (``tpc_refit_full_ce``).  Returns (ok, chain_hits, chain_pieces, par7, cov15)."""
        torch = self._torch
        o, st = outputs
        K = max(int(st.max_tracks), 1)
        if out is None:
            e = lambda shape, dt: torch.empty(shape, dtype=dt, device=self.device)
            out = (e(K, torch.int32), e(K, torch.int32), e(K, torch.int32), e((K, 7), torch.float32), e((K, 15), torch.float32))
        m = Merged(*(t.data_ptr() for t in merged))
        r = FullFit(*(t.data_ptr() for t in out))
        fp = FullFitParams(*(float(v) for v in full_params))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        if ce_merged is None:
            rc = self.lib.tpc_refit_full(self.handle, C.byref(fp), C.byref(st), C.byref(m), C.c_void_p(s.cuda_stream), C.byref(r))
        else:
            cm = CeMerged(*(t.data_ptr() for t in ce_merged))
            rc = self.lib.tpc_refit_full_ce(self.handle, C.byref(fp), C.byref(st), C.byref(m), C.byref(cm), C.c_void_p(s.cuda_stream), C.byref(r))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_refit_full")
        return out

    def tpc_compress_tracks(self, outputs, n_clusters: int, reject_q_pt: float = 1.0 / 0.15, step_y: float = 0.025, step_z: float = 0.025,
                            out=None, stream=None):
        """C11 on the DEVICE track outputs (allocated with ``hit_coords=True``); returns (reject uint8[n_clusters],
        ok int32[max_tracks], res_y int16[max_track_hits], res_z int16[max_track_hits])."""
        torch = self._torch
        o, st = outputs
        K, H = max(int(st.max_tracks), 1), max(int(st.max_track_hits), 1)
        if out is None:
            e = lambda n, dt: torch.empty(n, dtype=dt, device=self.device)
            out = (e(max(int(n_clusters), 1), torch.uint8), e(K, torch.int32), e(H, torch.int16), e(H, torch.int16))
        cp = CompressParams(float(reject_q_pt), float(step_y), float(step_z))
        co = Compressed(*(t.data_ptr() for t in out))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self.lib.tpc_compress_tracks(self.handle, C.byref(cp), C.byref(st), int(n_clusters), C.c_void_p(s.cuda_stream), C.byref(co))
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_compress_tracks")
        return out

    def tpc_vertex_time(self, n_tracks, par7, stream=None):
        """C9: (ok, vertex_time [time bins], vertex_y [cm]) of the DEVICE states ``par7`` (float32[K, 7]); ``n_tracks`` is the
        1-element device tensor written by ``tpc_track_timeframe``."""
        torch = self._torch
        K = int(par7.shape[0])
        ok = torch.empty(max(K, 1), dtype=torch.int32, device=self.device)
        vt, vy = (torch.empty(max(K, 1), dtype=torch.float32, device=self.device) for _ in range(2))
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        rc = self.lib.tpc_vertex_time(self.handle, n_tracks.data_ptr(), K, par7.data_ptr(), C.c_void_p(s.cuda_stream),
                                      ok.data_ptr(), vt.data_ptr(), vy.data_ptr())
        if rc != TPC_OK:
            raise TpcError(rc, "tpc_vertex_time")
        return ok, vt, vy

    def merge_scratch_bytes(self, max_tracks: int) -> int:
        return int(self.lib.tpc_merge_scratch_bytes(self.handle, int(max_tracks)))

    def last_merge_launches(self) -> int:
        return int(self.lib.tpc_merge_last_launches(self.handle))

    def step_ms(self) -> dict:
        buf = (C.c_float * 32)()
        k = self.lib.tpc_tracker_step_ms(self.handle, buf, 32)
        if k < 0:
            raise TpcError(k, "tpc_tracker_step_ms")
        return {self.lib.tpc_tracker_step_name(i).decode(): float(buf[i]) for i in range(k)}

    def last_launches(self) -> int:
        return int(self.lib.tpc_tracker_last_launches(self.handle))

    def work_counters(self, stream=None) -> dict:
        s = stream if stream is not None else self._torch.cuda.current_stream(self.device)
        buf = (C.c_int64 * 22)()
        k = self.lib.tpc_tracker_work_counters(self.handle, C.c_void_p(s.cuda_stream), buf, 22)
        if k < 0:
            raise TpcError(k, "tpc_tracker_work_counters")
        names = ("tracklets", "start_hits", "invalid_clusters", "row_steps", "updates", "candidates")
        out = {nm: int(buf[i]) for i, nm in enumerate(names)}
        for p, ph in enumerate(("fit_up", "follow_up", "fit_down", "follow_down")):
            out[ph] = {nm: int(buf[6 + 3 * p + i]) for i, nm in enumerate(("row_steps", "updates", "candidates"))}
        out["rare_paths"] = {"refit_replays": int(buf[18]), "refits_without_update": int(buf[19]), "search_ties": int(buf[20]),
                             "searches_in_global_memory": int(buf[21])}
        return out

    def arena_plan(self) -> list:
        out, i = [], 0
        name, off, nb, a, b = C.c_char_p(), C.c_size_t(), C.c_size_t(), C.c_int32(), C.c_int32()
        while self.lib.tpc_tracker_arena_plan(self.handle, i, C.byref(name), C.byref(off), C.byref(nb), C.byref(a), C.byref(b)) > 0:
            out.append(dict(name=name.value.decode(), offset=off.value, bytes=nb.value, first_step=a.value, last_step=b.value))
            i += 1
        return out

    def tpc_tracker_destroy(self):
        if getattr(self, "handle", None) is not None and self.handle:
            self.lib.tpc_tracker_destroy(self.handle)
            self.handle = None

    close = tpc_tracker_destroy

    def __del__(self):
        try:
            self.tpc_tracker_destroy()
        except Exception:
            pass
