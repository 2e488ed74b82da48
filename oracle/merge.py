"""ORACLE -- test infrastructure only (ctypes binding of ``tpc_merge_oracle.cpp``, step C7: sector-boundary merging).

Same rules as ``oracle/__init__.py``: only tests, ``smoke()`` and ``bench.py``'s CPU legs may import it.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass

import numpy as np

from . import CXXFLAGS

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_merge_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpcmergeoracle.so")


class MergeParams(C.Structure):
    _fields_ = [("n_sectors", C.c_int32), ("x0_cm", C.c_float), ("row_pitch_cm", C.c_float),
                ("tan_half_sector", C.c_float), ("time_bin_cm", C.c_float),
                ("sin_phi_max", C.c_float), ("inv_R_per_qpt", C.c_float),
                ("cut_y_cm", C.c_float), ("cut_z_cm", C.c_float), ("cut_sin_phi", C.c_float), ("cut_q_pt", C.c_float),
                ("max_row_gap", C.c_int32), ("max_row_overlap", C.c_int32)]


def default_merge_params(n_sectors: int = 36) -> MergeParams:
    """DESIGN.md §3 C7 readings M4/M5: cuts 2 cm, 2 cm, 0.05, 0.5 (GeV/c)^-1; rows l_A - 1 .. l_A + 13."""
    return MergeParams(n_sectors, 85.0, 1.07, math.tan(math.radians(10.0)), 0.516, 0.95, 1.0 / 666.7,
                       2.0, 2.0, 0.05, 0.5, 12, 2)


class CeParams(C.Structure):
    """``orc_ce_params`` (C10: merging across the central electrode)."""
    _fields_ = [("n_sectors", C.c_int32), ("n_rows", C.c_int32), ("x0_cm", C.c_float), ("row_pitch_cm", C.c_float),
                ("time_bin_cm", C.c_float), ("sin_phi_max", C.c_float), ("inv_R_per_qpt", C.c_float),
                ("cut_y_cm", C.c_float), ("cut_z_cm", C.c_float), ("cut_sin_phi", C.c_float), ("cut_q_pt", C.c_float),
                ("cut_dzds", C.c_float), ("max_row_gap", C.c_int32), ("max_row_overlap", C.c_int32)]


def default_ce_params(n_sectors: int = 36) -> CeParams:
    """DESIGN.md §3 C10 reading CE5: the cuts of C7 plus 0.1 on the mirrored dz/ds."""
    return CeParams(n_sectors, 152, 85.0, 1.07, 0.516, 0.95, 1.0 / 666.7, 2.0, 2.0, 0.05, 0.5, 0.1, 12, 2)


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
        L.orc_merge.argtypes = [C.POINTER(MergeParams), C.c_int64] + [vp] * 9
        L.orc_merge.restype = C.c_int64
        L.orc_merge_rotate.argtypes = [C.POINTER(MergeParams), vp, C.c_int32]
        L.orc_merge_rotate.restype = None
        L.orc_merge_transport.argtypes = [C.POINTER(MergeParams), vp, C.c_float]
        L.orc_merge_transport.restype = C.c_int
        L.orc_vertex_time.argtypes = [C.POINTER(MergeParams), C.c_int64, vp, vp, vp, vp]
        L.orc_vertex_time.restype = None
        L.orc_merge_ce.argtypes = [C.POINTER(CeParams), C.c_int64] + [vp] * 8
        L.orc_merge_ce.restype = C.c_int64
        _lib = L
    return _lib


@dataclass
class MergeResult:
    n_links: int
    next: np.ndarray      # int32[n] track index of the outer continuation, -1 = none
    prev: np.ndarray      # int32[n] track index of the inner piece, -1 = none
    root: np.ndarray      # int32[n] first piece of the chain (i itself for an unmerged track)
    best_d2: np.ndarray   # float32[n] d2 of out[A] (-1 = no candidate), for diagnostics


def merge(p: MergeParams, seed, sector, first_row, last_row, par) -> MergeResult:
    """C7 on host arrays; ``par`` is float32[n, 7] = (x, y, z_rel, sin_phi, dzds, q_pt, time_ref)."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    seed, sector, first_row, last_row = (a(v, np.int32) for v in (seed, sector, first_row, last_row))
    par = a(par, np.float32).reshape(-1, 7)
    n = int(seed.shape[0])
    nxt, prv, root = (np.empty(n, np.int32) for _ in range(3))
    d2 = np.empty(n, np.float32)
    k = lib().orc_merge(C.byref(p), n, seed.ctypes.data, sector.ctypes.data, first_row.ctypes.data,
                        last_row.ctypes.data, par.ctypes.data, nxt.ctypes.data, prv.ctypes.data, root.ctypes.data,
                        d2.ctypes.data)
    return MergeResult(int(k), nxt, prv, root, d2)


def rotate(p: MergeParams, state6, side_sign: int) -> np.ndarray:
    st = np.array(state6, np.float32)
    lib().orc_merge_rotate(C.byref(p), st.ctypes.data, int(side_sign))
    return st


def transport_state(p: MergeParams, state6, xn: float):
    st = np.array(state6, np.float32)
    ok = lib().orc_merge_transport(C.byref(p), st.ctypes.data, float(xn))
    return bool(ok), st


def vertex_time(p: MergeParams, par):
    """C9: (ok, vertex_time [time bins], vertex_y [cm]) of every state in ``par`` (float32[n, 7]) transported to the beam line."""
    par = np.ascontiguousarray(par, np.float32).reshape(-1, 7)
    n = int(par.shape[0])
    ok, t, y = np.zeros(n, np.int32), np.zeros(n, np.float32), np.zeros(n, np.float32)
    lib().orc_vertex_time(C.byref(p), n, par.ctypes.data, ok.ctypes.data, t.ctypes.data, y.ctypes.data)
    return ok, t, y


@dataclass
class CeResult:
    n_links: int
    next: np.ndarray      # int32[n] the continuation of track i behind the central electrode (mirror sector), -1 = none
    prev: np.ndarray      # int32[n]
    t_ce: np.ndarray      # float32[n] time coordinate of the crossing [time bins] for linked i, else 0


def merge_ce(p: CeParams, seed, sector, first_row, last_row, par) -> CeResult:
    """C10 on host arrays; ``par`` is float32[n, 7] = (x, y, z_rel, sin_phi, dzds, q_pt, time_ref)."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    seed, sector, first_row, last_row = (a(v, np.int32) for v in (seed, sector, first_row, last_row))
    par = a(par, np.float32).reshape(-1, 7)
    n = int(seed.shape[0])
    nxt, prv = (np.empty(n, np.int32) for _ in range(2))
    tce = np.empty(n, np.float32)
    k = lib().orc_merge_ce(C.byref(p), n, seed.ctypes.data, sector.ctypes.data, first_row.ctypes.data, last_row.ctypes.data,
                           par.ctypes.data, nxt.ctypes.data, prv.ctypes.data, tce.ctypes.data)
    return CeResult(int(k), nxt, prv, tce)
