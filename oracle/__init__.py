"""ORACLE -- test infrastructure only (ctypes binding of ``tpc_oracle.cpp``).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It shares no code with ``paper_2102_08862_b200/csrc`` and never imports the product
package's CUDA binding.  See the header of ``tpc_oracle.cpp`` for what it follows and what pins it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpcoracle.so")

# -ffp-contract=off: no FMA contraction; no -ffast-math; x86-64 SSE2 scalar fp32 (no x87 excess precision)
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]


class Geometry(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("x0_cm", C.c_float),
                ("row_pitch_cm", C.c_float), ("pad_pitch_cm", C.c_float), ("tan_half_sector", C.c_float),
                ("time_bin_cm", C.c_float), ("drift_len_cm", C.c_float), ("max_time_bin", C.c_float)]


class Params(C.Structure):
    _fields_ = [("win_slope", C.c_float), ("win_const", C.c_float), ("chi2_cut", C.c_float),
                ("miss_limit", C.c_int32), ("min_hits", C.c_int32),
                ("sigma_y_cm", C.c_float), ("sigma_z_cm", C.c_float),
                ("slope_y_max", C.c_float), ("slope_z_max", C.c_float), ("seed_min_hits", C.c_int32),
                ("sin_phi_max", C.c_float), ("inv_R_per_qpt", C.c_float),
                ("c0_y2", C.c_float), ("c0_s2", C.c_float), ("c0_k2", C.c_float), ("c0_z2", C.c_float),
                ("c0_t2", C.c_float), ("brute_force", C.c_int32)]


def default_geometry(n_sectors: int = 36, max_time_bin: float = 487.0) -> Geometry:
    """BASELINE.json L7: 152 rows at 85.0 + 1.07 r cm, 0.5 cm pads, +-10 deg sectors, 0.516 cm time bins."""
    import math
    return Geometry(n_sectors, 152, 85.0, 1.07, 0.5, math.tan(math.radians(10.0)), 0.516, 250.0, max_time_bin)


def default_params(sigma_y: float = 0.08, sigma_z: float = 0.12) -> Params:
    """BASELINE.json L7 cuts + the [proposed] readings of SURVEY.md §8(c) / DESIGN.md."""
    return Params(win_slope=0.05, win_const=0.5, chi2_cut=9.0, miss_limit=10, min_hits=30,
                  sigma_y_cm=sigma_y, sigma_z_cm=sigma_z, slope_y_max=1.0, slope_z_max=1.5,
                  seed_min_hits=3, sin_phi_max=0.95, inv_R_per_qpt=1.0 / 666.7,
                  c0_y2=1.0, c0_s2=0.1, c0_k2=100.0, c0_z2=1.0, c0_t2=0.1, brute_force=0)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", *CXXFLAGS, "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp = C.c_void_p
        L.orc_track.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, vp, C.c_int64, C.POINTER(vp)]
        L.orc_track.restype = C.c_int
        for nm in ("orc_n_tracklets", "orc_n_tracks", "orc_n_track_hits"):
            getattr(L, nm).argtypes = [vp]
            getattr(L, nm).restype = C.c_int64
        L.orc_copy_links.argtypes = [vp] * 6
        L.orc_copy_tracklets.argtypes = [vp] * 8
        L.orc_copy_tracks.argtypes = [vp] * 10
        L.orc_copy_stats.argtypes = [vp, vp]
        L.orc_free.argtypes = [vp]
        L.orc_transport.argtypes = [C.POINTER(Params), vp, vp, C.c_float]
        L.orc_transport.restype = C.c_int
        L.orc_update.argtypes = [vp, vp, C.c_float, C.c_float, C.c_float, C.c_float]
        L.orc_tables.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, vp, vp]
        L.orc_refit_chains.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, vp, C.c_int64] + [vp] * 12
        L.orc_refit_chains.restype = None
        L.orc_compress_tracks.argtypes = [C.POINTER(Geometry), C.POINTER(Params), C.c_float, C.c_float, C.c_float, vp, vp, vp, C.c_int64,
                                          C.c_int64] + [vp] * 9
        L.orc_compress_tracks.restype = None
        L.orc_decompress_tracks.argtypes = [C.POINTER(Geometry), C.POINTER(Params), C.c_float, C.c_float, C.c_int64] + [vp] * 10
        L.orc_decompress_tracks.restype = None
        L.orc_rotate_with_cov.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, C.c_int32]
        L.orc_rotate_with_cov.restype = C.c_int
        L.orc_refit_full.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, vp, vp, C.c_int64] + [vp] * 12
        L.orc_refit_full.restype = None
        L.orc_refit_full_ce.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, vp, vp, C.c_int64] + [vp] * 15
        L.orc_refit_full_ce.restype = None
        L.orc_full_reflect.argtypes = [vp, vp, C.c_float, C.c_float, C.c_float, C.c_float]
        L.orc_full_reflect.restype = None
        L.orc_full_step.argtypes = [C.POINTER(Params), vp, vp, vp, C.c_float]
        L.orc_full_step.restype = C.c_int
        L.orc_full_update.argtypes = [vp, vp, C.c_float, C.c_float, C.c_float, C.c_float]
        L.orc_full_update.restype = None
        L.orc_full_rotate.argtypes = [C.POINTER(Geometry), C.POINTER(Params), vp, vp, C.c_int32]
        L.orc_full_rotate.restype = C.c_int
        for nm in ("orc_copy_links", "orc_copy_tracklets", "orc_copy_tracks", "orc_copy_stats", "orc_free",
                   "orc_update", "orc_tables"):
            getattr(L, nm).restype = None
        _lib = L
    return _lib


STAT_NAMES = ("s_ingest", "s_finder", "s_cleaner_start", "s_constructor", "s_selector", "finder_candidates",
              "finder_pairs", "transports", "searches", "search_candidates", "updates", "invalid_clusters",
              "start_hits")

PAR_NAMES = ("x", "y", "z_rel", "sin_phi", "dzds", "q_pt", "time_ref")


@dataclass
class Result:
    n: int
    up_raw: np.ndarray
    down_raw: np.ndarray
    link_up: np.ndarray        # cleaned, by original index, -1 = none
    link_down: np.ndarray
    is_start_hit: np.ndarray   # uint8[n]
    tl_seed: np.ndarray        # tracklets: one per start hit, in ascending start-hit index
    tl_n_hits: np.ndarray
    tl_first_row: np.ndarray
    tl_last_row: np.ndarray
    tl_row_hit: np.ndarray     # int32[n_tracklets, n_rows]
    tl_par: np.ndarray         # float32[n_tracklets, 7]
    tl_cov: np.ndarray         # float32[n_tracklets, 9]
    tr_seed: np.ndarray        # tracks
    tr_sector: np.ndarray
    tr_first_row: np.ndarray
    tr_last_row: np.ndarray
    tr_n_hits: np.ndarray
    tr_hit_offset: np.ndarray
    tr_par: np.ndarray
    tr_cov: np.ndarray
    tr_hit_index: np.ndarray   # original cluster indices, ascending row, per track contiguous
    stats: dict

    def track_hits(self, i: int) -> np.ndarray:
        o = int(self.tr_hit_offset[i])
        return self.tr_hit_index[o:o + int(self.tr_n_hits[i])]


def track(geom: Geometry, params: Params, row, pad, time) -> Result:
    """Run the whole path (C1..C6) on host fp32 arrays."""
    L = lib()
    row = np.ascontiguousarray(row, np.float32)
    pad = np.ascontiguousarray(pad, np.float32)
    time = np.ascontiguousarray(time, np.float32)
    n = int(row.shape[0])
    assert pad.shape[0] == n and time.shape[0] == n
    h = C.c_void_p()
    rc = L.orc_track(C.byref(geom), C.byref(params), row.ctypes.data, pad.ctypes.data, time.ctypes.data, n, C.byref(h))
    if rc != 0:
        raise ValueError("orc_track rejected its arguments")
    try:
        nr = geom.n_rows
        i32 = lambda *s: np.empty(s, np.int32)
        up_raw, down_raw, up, down = i32(n), i32(n), i32(n), i32(n)
        st = np.empty(n, np.uint8)
        L.orc_copy_links(h, up_raw.ctypes.data, down_raw.ctypes.data, up.ctypes.data, down.ctypes.data, st.ctypes.data)
        nt = L.orc_n_tracklets(h)
        ts, tn, tf, tl, trh = i32(nt), i32(nt), i32(nt), i32(nt), i32(nt, nr)
        tp, tc = np.empty((nt, 7), np.float32), np.empty((nt, 9), np.float32)
        L.orc_copy_tracklets(h, ts.ctypes.data, tn.ctypes.data, tf.ctypes.data, tl.ctypes.data, trh.ctypes.data,
                             tp.ctypes.data, tc.ctypes.data)
        nk, nh = L.orc_n_tracks(h), L.orc_n_track_hits(h)
        ks, kc, kf, kl, kn = i32(nk), i32(nk), i32(nk), i32(nk), i32(nk)
        ko = np.empty(nk, np.int64)
        kp, kv = np.empty((nk, 7), np.float32), np.empty((nk, 9), np.float32)
        kh = i32(nh)
        L.orc_copy_tracks(h, ks.ctypes.data, kc.ctypes.data, kf.ctypes.data, kl.ctypes.data, kn.ctypes.data,
                          ko.ctypes.data, kp.ctypes.data, kv.ctypes.data, kh.ctypes.data)
        s16 = np.zeros(16, np.float64)
        L.orc_copy_stats(h, s16.ctypes.data)
        stats = {k: float(s16[i]) for i, k in enumerate(STAT_NAMES)}
        return Result(n, up_raw, down_raw, up, down, st, ts, tn, tf, tl, trh, tp, tc,
                      ks, kc, kf, kl, kn, ko, kp, kv, kh, stats)
    finally:
        L.orc_free(h)


def transport(params: Params, state6, cov9, xn: float):
    """One call of the oracle's transport (pins K1, K2).  Returns (ok, state6, cov9)."""
    st = np.array(state6, np.float32)
    cv = np.array(cov9, np.float32)
    rc = lib().orc_transport(C.byref(params), st.ctypes.data, cv.ctypes.data, float(xn))
    return rc == 0, st, cv


def update(state6, cov9, ym: float, zm: float, ry: float, rz: float):
    """One call of the oracle's Kalman update (pin K3)."""
    st = np.array(state6, np.float32)
    cv = np.array(cov9, np.float32)
    lib().orc_update(st.ctypes.data, cv.ctypes.data, float(ym), float(zm), float(ry), float(rz))
    return st, cv


def tables(geom: Geometry, params: Params):
    """Geometry tables and derived constants as the oracle computes them (pin G1)."""
    nr = geom.n_rows
    x = np.empty(nr, np.float32)
    npads = np.empty(nr, np.int32)
    cr = np.empty(nr, np.float32)
    k = np.empty(8, np.float32)
    lib().orc_tables(C.byref(geom), C.byref(params), x.ctypes.data, npads.ctypes.data, cr.ctypes.data, k.ctypes.data)
    return x, npads, cr, dict(W1=k[0], Ay=k[1], Az=k[2], wy=k[3], wz=k[4], ry=k[5], rz=k[6])


def refit_chains(geom: Geometry, params: Params, row, pad, time, res: "Result", nxt, prv):
    """C8: refit of the chains linked by C7 (``oracle.merge``).  Returns (ok, chain_hits, chain_pieces, par[n,7], cov[n,9])."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    row, pad, time = a(row, np.float32), a(pad, np.float32), a(time, np.float32)
    nxt, prv = a(nxt, np.int32), a(prv, np.int32)
    n = int(len(res.tr_seed))
    ok, ch, cp = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32)
    rp, rc = np.zeros((n, 7), np.float32), np.zeros((n, 9), np.float32)
    sec, nh, off = a(res.tr_sector, np.int32), a(res.tr_n_hits, np.int32), a(res.tr_hit_offset, np.int64)
    hi, par = a(res.tr_hit_index, np.int32), a(res.tr_par, np.float32)
    lib().orc_refit_chains(C.byref(geom), C.byref(params), row.ctypes.data, pad.ctypes.data, time.ctypes.data, n,
                           sec.ctypes.data, nh.ctypes.data, off.ctypes.data, hi.ctypes.data, par.ctypes.data,
                           nxt.ctypes.data, prv.ctypes.data, ok.ctypes.data, ch.ctypes.data, cp.ctypes.data,
                           rp.ctypes.data, rc.ctypes.data)
    return ok, ch, cp, rp, rc


def rotate_with_cov(geom: Geometry, params: Params, state6, cov9, q: int):
    """C8 rotation of state and covariance by q * 20 degrees (pin F-J).  Returns (ok, state6, cov9)."""
    st = np.array(state6, np.float32)
    cv = np.array(cov9, np.float32)
    rc = lib().orc_rotate_with_cov(C.byref(geom), C.byref(params), st.ctypes.data, cv.ctypes.data, int(q))
    return rc == 0, st, cv


# C12 material of the drift gas (DESIGN.md §3 C12 reading FF3): (1 / radiation length [1/cm], dE/dx of a minimum-ionising
# particle [GeV/cm], particle mass [GeV], relative width of the energy loss)
DEFAULT_FULL_PARAMS = (1.0 / 3.0e4, 1.7e-6, 0.13957, 0.1)


def refit_full(geom: Geometry, params: Params, row, pad, time, res: "Result", nxt, prv, full_params=DEFAULT_FULL_PARAMS):
    """C12: full-covariance refit with material of every chain root.  Returns (ok, chain_hits, chain_pieces, par[n,7], cov[n,15])."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    row, pad, time = a(row, np.float32), a(pad, np.float32), a(time, np.float32)
    nxt, prv = a(nxt, np.int32), a(prv, np.int32)
    n = int(len(res.tr_seed))
    ok, ch, cp = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32)
    rp, rc = np.zeros((n, 7), np.float32), np.zeros((n, 15), np.float32)
    sec, nh, off = a(res.tr_sector, np.int32), a(res.tr_n_hits, np.int32), a(res.tr_hit_offset, np.int64)
    hi, par = a(res.tr_hit_index, np.int32), a(res.tr_par, np.float32)
    f4 = np.array(full_params, np.float32)
    lib().orc_refit_full(C.byref(geom), C.byref(params), f4.ctypes.data, row.ctypes.data, pad.ctypes.data, time.ctypes.data, n,
                         sec.ctypes.data, nh.ctypes.data, off.ctypes.data, hi.ctypes.data, par.ctypes.data,
                         nxt.ctypes.data, prv.ctypes.data, ok.ctypes.data, ch.ctypes.data, cp.ctypes.data,
                         rp.ctypes.data, rc.ctypes.data)
    return ok, ch, cp, rp, rc


def refit_full_ce(geom: Geometry, params: Params, row, pad, time, res: "Result", nxt, prv, ce_next, ce_prev, t_ce,
                  full_params=DEFAULT_FULL_PARAMS):
    """C12 over chains that may continue behind the central electrode (C10's links; reading FF8).  Returns like refit_full."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    row, pad, time = a(row, np.float32), a(pad, np.float32), a(time, np.float32)
    nxt, prv, cn, cp_, tc = a(nxt, np.int32), a(prv, np.int32), a(ce_next, np.int32), a(ce_prev, np.int32), a(t_ce, np.float32)
    n = int(len(res.tr_seed))
    ok, ch, cp = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32)
    rp, rc = np.zeros((n, 7), np.float32), np.zeros((n, 15), np.float32)
    sec, nh, off = a(res.tr_sector, np.int32), a(res.tr_n_hits, np.int32), a(res.tr_hit_offset, np.int64)
    hi, par = a(res.tr_hit_index, np.int32), a(res.tr_par, np.float32)
    f4 = np.array(full_params, np.float32)
    lib().orc_refit_full_ce(C.byref(geom), C.byref(params), f4.ctypes.data, row.ctypes.data, pad.ctypes.data, time.ctypes.data, n,
                            sec.ctypes.data, nh.ctypes.data, off.ctypes.data, hi.ctypes.data, par.ctypes.data,
                            nxt.ctypes.data, prv.ctypes.data, cn.ctypes.data, cp_.ctypes.data, tc.ctypes.data,
                            ok.ctypes.data, ch.ctypes.data, cp.ctypes.data, rp.ctypes.data, rc.ctypes.data)
    return ok, ch, cp, rp, rc


def full_step(params: Params, state6, cov15, xn: float, full_params=DEFAULT_FULL_PARAMS):
    """One transport + material step of C12 (pins FF-*).  Returns (ok, state6, cov15)."""
    st, cv, f4 = np.array(state6, np.float32), np.array(cov15, np.float32), np.array(full_params, np.float32)
    rc = lib().orc_full_step(C.byref(params), f4.ctypes.data, st.ctypes.data, cv.ctypes.data, float(xn))
    return rc == 0, st, cv


def full_rotate(geom: Geometry, params: Params, state6, cov15, q: int):
    """C12 rotation of state and covariance by q * 20 degrees (pin FF-R).  Returns (ok, state6, cov15)."""
    st, cv = np.array(state6, np.float32), np.array(cov15, np.float32)
    rc = lib().orc_full_rotate(C.byref(geom), C.byref(params), st.ctypes.data, cv.ctypes.data, int(q))
    return rc == 0, st, cv


def full_reflect(state6, cov15, tc: float, tref_b: float, tref_e: float, Z: float = 0.516):
    """C12's reflection at the central electrode (pin FF-CE-R).  Returns (state6, cov15)."""
    st, cv = np.array(state6, np.float32), np.array(cov15, np.float32)
    lib().orc_full_reflect(st.ctypes.data, cv.ctypes.data, float(tc), float(tref_b), float(tref_e), float(Z))
    return st, cv


def full_update(state6, cov15, ym: float, zm: float, ry: float, rz: float):
    """The two scalar updates of C12 with one hit."""
    st, cv = np.array(state6, np.float32), np.array(cov15, np.float32)
    lib().orc_full_update(st.ctypes.data, cv.ctypes.data, float(ym), float(zm), float(ry), float(rz))
    return st, cv


DEFAULT_REJECT_QPT, DEFAULT_STEP_Y, DEFAULT_STEP_Z = 1.0 / 0.15, 0.025, 0.025      # DESIGN.md §3 C11 readings R11-1, R11-3


def compress_tracks(geom: Geometry, params: Params, row, pad, time, res: "Result", reject_qpt: float = DEFAULT_REJECT_QPT,
                    step_y: float = DEFAULT_STEP_Y, step_z: float = DEFAULT_STEP_Z):
    """C11: (reject uint8[n_clusters], ok int32[n_tracks], qy int16[n_track_hits], qz int16[n_track_hits])."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    row, pad, time = a(row, np.float32), a(pad, np.float32), a(time, np.float32)
    n, k, nh = int(row.shape[0]), int(len(res.tr_seed)), int(len(res.tr_hit_index))
    reject, ok = np.zeros(n, np.uint8), np.zeros(k, np.int32)
    qy, qz = np.zeros(nh, np.int16), np.zeros(nh, np.int16)
    nhits, off, hi = a(res.tr_n_hits, np.int32), a(res.tr_hit_offset, np.int64), a(res.tr_hit_index, np.int32)
    par, cov = a(res.tr_par, np.float32), a(res.tr_cov, np.float32)
    lib().orc_compress_tracks(C.byref(geom), C.byref(params), float(reject_qpt), float(step_y), float(step_z), row.ctypes.data,
                              pad.ctypes.data, time.ctypes.data, n, k, nhits.ctypes.data, off.ctypes.data, hi.ctypes.data,
                              par.ctypes.data, cov.ctypes.data, reject.ctypes.data, ok.ctypes.data, qy.ctypes.data, qz.ctypes.data)
    return reject, ok, qy, qz


def decompress_tracks(geom: Geometry, params: Params, res: "Result", hit_row, ok, qy, qz, step_y: float = DEFAULT_STEP_Y,
                      step_z: float = DEFAULT_STEP_Z):
    """The C11 decoder (pins only): (y [cm], z relative to the track's time_ref [cm]) of every hit of the tracks with ok == 1."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    k, nh = int(len(res.tr_seed)), int(len(res.tr_hit_index))
    y, z = np.full(nh, np.nan, np.float32), np.full(nh, np.nan, np.float32)
    nhits, off = a(res.tr_n_hits, np.int32), a(res.tr_hit_offset, np.int64)
    par, cov, hr = a(res.tr_par, np.float32), a(res.tr_cov, np.float32), a(hit_row, np.uint8)
    ok, qy, qz = a(ok, np.int32), a(qy, np.int16), a(qz, np.int16)
    lib().orc_decompress_tracks(C.byref(geom), C.byref(params), float(step_y), float(step_z), k, nhits.ctypes.data, off.ctypes.data,
                                hr.ctypes.data, par.ctypes.data, cov.ctypes.data, ok.ctypes.data, qy.ctypes.data, qz.ctypes.data,
                                y.ctypes.data, z.ctypes.data)
    return y, z
