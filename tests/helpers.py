"""Small shared helpers for the tests: build cluster arrays from analytic tracks (inputs only)."""
from __future__ import annotations

import math

import numpy as np

N_ROWS = 152
X0, PITCH, PAD_PITCH, ZBIN = 85.0, 1.07, 0.5, 0.516
TAN10 = math.tan(math.radians(10.0))


def row_x(r):
    return X0 + PITCH * np.asarray(r, dtype=np.float64)


def n_pads(r):
    return np.floor(2.0 * row_x(r) * TAN10 / PAD_PITCH).astype(np.int64)


def clusters_from_xyz(rows, y, z_time_cm, sector=0):
    """fp32 (row, pad, time) from local y [cm] and the time-derived coordinate [cm] at integer rows."""
    rows = np.asarray(rows, np.int64)
    pad = np.asarray(y, np.float64) / PAD_PITCH + 0.5 * (n_pads(rows) - 1)
    time = np.asarray(z_time_cm, np.float64) / ZBIN
    return ((sector * N_ROWS + rows).astype(np.float32), pad.astype(np.float32), time.astype(np.float32))


def concat(parts):
    return tuple(np.concatenate([p[i] for p in parts]) for i in range(3))
