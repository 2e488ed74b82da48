"""ORACLE -- test infrastructure only (ctypes binding of ``tpc_cluster_oracle.cpp``, step C0: the TPC cluster finder).

Same rules as ``oracle/__init__.py``: only tests, ``smoke()`` and ``bench.py``'s CPU legs may import it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

from . import CXXFLAGS

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_cluster_oracle.cpp")
_LIB = os.path.join(_HERE, "libtpcclusteroracle.so")

DEFAULT_PEAK_THRESHOLD = 8.0        # DESIGN.md §3 C0 reading D4


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
        L.orc_find_clusters.argtypes = [C.c_int64, vp, vp, vp, vp, C.c_float, C.POINTER(vp)]
        L.orc_find_clusters.restype = C.c_int
        L.orc_cf_n.argtypes = [vp]
        L.orc_cf_n.restype = C.c_int64
        L.orc_cf_copy.argtypes = [vp] * 6
        L.orc_cf_copy.restype = None
        L.orc_cf_free.argtypes = [vp]
        L.orc_cf_free.restype = None
        _lib = L
    return _lib


@dataclass
class Clusters:
    row: np.ndarray      # float32[n]  sector*n_rows + pad row (the tracker's input encoding)
    pad: np.ndarray      # float32[n]
    time: np.ndarray     # float32[n]
    charge: np.ndarray   # float32[n]
    peak: np.ndarray     # int64[n]    input index of the peak sample

    @property
    def n(self) -> int:
        return int(self.peak.shape[0])


def find_clusters(row, pad, time, adc, peak_threshold: float = DEFAULT_PEAK_THRESHOLD) -> Clusters:
    """C0 on host arrays: int32 (row, pad, time) and float32 adc, sorted by (row, time, pad)."""
    a = lambda v, t: np.ascontiguousarray(v, t)
    row, pad, time, adc = a(row, np.int32), a(pad, np.int32), a(time, np.int32), a(adc, np.float32)
    n = int(adc.shape[0])
    h = C.c_void_p()
    rc = lib().orc_find_clusters(n, row.ctypes.data, pad.ctypes.data, time.ctypes.data, adc.ctypes.data, float(peak_threshold), C.byref(h))
    if rc != 0:
        raise ValueError("orc_find_clusters rejected its input (not sorted by (row, time, pad) or out of range)" if rc == -2 else "orc_find_clusters: bad arguments")
    try:
        k = lib().orc_cf_n(h)
        f = lambda: np.empty(k, np.float32)
        r, p, t, q = f(), f(), f(), f()
        pk = np.empty(k, np.int64)
        lib().orc_cf_copy(h, r.ctypes.data, p.ctypes.data, t.ctypes.data, q.ctypes.data, pk.ctypes.data)
        return Clusters(r, p, t, q, pk)
    finally:
        lib().orc_cf_free(h)
