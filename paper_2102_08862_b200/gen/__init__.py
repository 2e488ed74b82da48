"""Seeded synthetic TPC time-frame generator (ctypes binding of ``tfgen.cpp``).

Stands in for the paper's Monte-Carlo time frames (§2), which are not available.
The recipe is BASELINE.json configs[0..4] and SURVEY.md §8(d); DESIGN.md §"Input recipe" states it.
This module is the ONLY code shared by the oracle tests and the CUDA path: it produces inputs and
truth labels and contains none of the tracker's arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tfgen.cpp")
_LIB = os.path.join(_HERE, "libtfgen.so")


class GenConfig(C.Structure):
    """Mirror of ``struct tfgen_config``."""

    _fields_ = [
        ("n_sectors", C.c_int32), ("n_rows", C.c_int32),
        ("x0_cm", C.c_double), ("row_pitch_cm", C.c_double), ("pad_pitch_cm", C.c_double),
        ("half_sector_deg", C.c_double), ("time_bin_cm", C.c_double), ("drift_len_cm", C.c_double),
        ("v_drift_cm_us", C.c_double), ("frame_us", C.c_double), ("rate_khz", C.c_double),
        ("fixed_tracks", C.c_int32), ("max_tracks", C.c_int32),
        ("sigma_y_cm", C.c_double), ("sigma_z_cm", C.c_double),
        ("dropout", C.c_double), ("noise_frac", C.c_double),
        ("pt_min", C.c_double), ("pt_mean", C.c_double), ("pt_cap", C.c_double),
        ("eta_max", C.c_double), ("zv_sigma_cm", C.c_double), ("radius_per_pt", C.c_double),
        ("max_turns", C.c_int32), ("shuffle", C.c_int32),
        ("seed", C.c_uint64), ("n_threads", C.c_int32), ("reserved", C.c_int32),
    ]


class _Track(C.Structure):
    _fields_ = [("collision", C.c_int32), ("charge_sense", C.c_int32), ("t0_us", C.c_double),
                ("z_v", C.c_double), ("phi0", C.c_double), ("eta", C.c_double), ("pt", C.c_double)]


TRACK_DTYPE = np.dtype([("collision", "<i4"), ("charge_sense", "<i4"), ("t0_us", "<f8"),
                        ("z_v", "<f8"), ("phi0", "<f8"), ("eta", "<f8"), ("pt", "<f8")])
assert TRACK_DTYPE.itemsize == C.sizeof(_Track)


def build(force: bool = False) -> str:
    """Compile ``libtfgen.so`` in-tree with g++ if it is missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.tfgen_generate.argtypes = [C.POINTER(GenConfig), C.POINTER(C.c_void_p)]
        lib.tfgen_generate.restype = C.c_int
        for name, rt in (("tfgen_n_clusters", C.c_int64), ("tfgen_n_real", C.c_int64),
                         ("tfgen_n_tracks", C.c_int64), ("tfgen_n_collisions", C.c_int32),
                         ("tfgen_max_time_bin", C.c_double)):
            getattr(lib, name).argtypes = [C.c_void_p]
            getattr(lib, name).restype = rt
        lib.tfgen_copy.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        lib.tfgen_copy.restype = C.c_int
        lib.tfgen_free.argtypes = [C.c_void_p]
        lib.tfgen_free.restype = None
        lib.tfgen_digitize.argtypes = [C.c_int64] + [C.c_void_p] * 4 + [C.c_int32, C.c_int32, C.c_void_p, C.c_int32, C.c_double, C.c_double,
                                       C.c_int32, C.c_int32, C.POINTER(C.c_void_p)]
        lib.tfgen_digitize.restype = C.c_int
        lib.tfgen_digits_n.argtypes = [C.c_void_p]
        lib.tfgen_digits_n.restype = C.c_int64
        lib.tfgen_digits_copy.argtypes = [C.c_void_p] * 5
        lib.tfgen_digits_copy.restype = None
        lib.tfgen_digits_free.argtypes = [C.c_void_p]
        lib.tfgen_digits_free.restype = None
        _lib = lib
    return _lib


def base_config(seed: int = 1) -> GenConfig:
    """The geometry and generator constants shared by all five configs (BASELINE.json L7)."""
    return GenConfig(
        n_sectors=36, n_rows=152, x0_cm=85.0, row_pitch_cm=1.07, pad_pitch_cm=0.5,
        half_sector_deg=10.0, time_bin_cm=0.516, drift_len_cm=250.0, v_drift_cm_us=2.58,
        frame_us=0.0, rate_khz=50.0, fixed_tracks=4000, max_tracks=4000,
        sigma_y_cm=0.08, sigma_z_cm=0.12, dropout=0.1, noise_frac=0.05,
        pt_min=0.1, pt_mean=0.5, pt_cap=20.0, eta_max=0.9, zv_sigma_cm=5.0, radius_per_pt=666.7,
        max_turns=5, shuffle=1, seed=seed, n_threads=0, reserved=0)


def preset(config_id: int, seed: int = 1, frame_us: float | None = None) -> GenConfig:
    """BASELINE.json configs[config_id].  ``frame_us`` overrides the frame length of the
    continuous-readout configs (used for bounded samples of configs[3]/[4])."""
    c = base_config(seed)
    if config_id == 0:      # single sector, one collision, exactly 300 tracks
        c.n_sectors, c.fixed_tracks = 1, 300
    elif config_id == 1:    # full TPC, one central collision of 4000 tracks
        pass
    elif config_id == 2:    # 2 ms continuous readout
        c.fixed_tracks, c.frame_us = 0, 2000.0
    elif config_id == 3:    # 10 ms continuous readout
        c.fixed_tracks, c.frame_us = 0, 10000.0
    elif config_id == 4:    # 10 ms high-occupancy stress frame
        c.fixed_tracks, c.frame_us = 0, 10000.0
        c.noise_frac, c.pt_min, c.dropout, c.sigma_y_cm, c.sigma_z_cm = 0.30, 0.05, 0.2, 0.15, 0.2
    else:
        raise ValueError("config_id must be 0..4")
    if frame_us is not None:
        if config_id < 2:
            raise ValueError("configs[0] and [1] are single collisions")
        c.frame_us = float(frame_us)
    return c


@dataclass
class TimeFrame:
    """fp32 SoA clusters (the tracker's input) plus truth labels (never passed to a tracker)."""

    config: GenConfig
    row: np.ndarray          # float32[n]  sector*n_rows + pad row, integer-valued
    pad: np.ndarray          # float32[n]
    time: np.ndarray         # float32[n]  time bins
    charge: np.ndarray       # float32[n]  unused by the path
    truth_track: np.ndarray  # int32[n]    global particle index, -1 = noise
    truth_arc: np.ndarray    # int16[n]    2*turn + returning
    tracks: np.ndarray       # TRACK_DTYPE[n_particles]
    n_real: int
    n_collisions: int
    max_time_bin: float
    extra: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.row.shape[0])


def generate(cfg: GenConfig, want_truth: bool = True) -> TimeFrame:
    lib = _load()
    h = C.c_void_p()
    rc = lib.tfgen_generate(C.byref(cfg), C.byref(h))
    if rc != 0:
        raise ValueError("tfgen_generate rejected the configuration")
    try:
        n = lib.tfgen_n_clusters(h)
        nt = lib.tfgen_n_tracks(h)
        row, pad, time, charge = (np.empty(n, np.float32) for _ in range(4))
        tt = np.empty(n if want_truth else 0, np.int32)
        ta = np.empty(n if want_truth else 0, np.int16)
        tr = np.empty(nt, TRACK_DTYPE)
        lib.tfgen_copy(h, row.ctypes.data, pad.ctypes.data, time.ctypes.data, charge.ctypes.data,
                       tt.ctypes.data if want_truth else None, ta.ctypes.data if want_truth else None,
                       tr.ctypes.data)
        return TimeFrame(cfg, row, pad, time, charge, tt, ta, tr, int(lib.tfgen_n_real(h)),
                         int(lib.tfgen_n_collisions(h)), float(lib.tfgen_max_time_bin(h)))
    finally:
        lib.tfgen_free(h)


@dataclass
class Digits:
    """Zero-suppressed ADC samples (the cluster finder's input), sorted by (sector_row, time bin, pad)."""

    row: np.ndarray    # int32[n]  sector*n_rows + pad row
    pad: np.ndarray    # int32[n]
    time: np.ndarray   # int32[n]  time bin
    adc: np.ndarray    # float32[n] integer-valued ADC count

    @property
    def n(self) -> int:
        return int(self.adc.shape[0])


def digitize(row, pad, time, charge, n_sectors: int, max_time_bin: float, n_rows: int = 152, sigma_pad: float = 0.45,
             sigma_time: float = 0.55, threshold: int = 3, n_threads: int = 0) -> Digits:
    """Clusters -> zero-suppressed samples (see ``tfgen_digitize``): every cluster deposits its charge on the 3 x 3 cells
    around it with Gaussian-integral weights, overlapping deposits add, ADC = floor, samples below ``threshold`` are dropped."""
    lib = _load()
    a = lambda v: np.ascontiguousarray(v, np.float32)
    row, pad, time, charge = a(row), a(pad), a(time), a(charge)
    x = 85.0 + 1.07 * np.arange(n_rows)
    npads = np.floor(2.0 * x * np.tan(np.radians(10.0)) / 0.5).astype(np.int32)
    h = C.c_void_p()
    rc = lib.tfgen_digitize(int(row.shape[0]), row.ctypes.data, pad.ctypes.data, time.ctypes.data, charge.ctypes.data,
                            int(n_sectors * n_rows), int(n_rows), npads.ctypes.data, int(max_time_bin), float(sigma_pad),
                            float(sigma_time), int(threshold), int(n_threads), C.byref(h))
    if rc != 0:
        raise ValueError("tfgen_digitize rejected its arguments")
    try:
        n = lib.tfgen_digits_n(h)
        r, p, t = (np.empty(n, np.int32) for _ in range(3))
        q = np.empty(n, np.float32)
        lib.tfgen_digits_copy(h, r.ctypes.data, p.ctypes.data, t.ctypes.data, q.ctypes.data)
        return Digits(r, p, t, q)
    finally:
        lib.tfgen_digits_free(h)
