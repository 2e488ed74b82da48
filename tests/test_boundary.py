"""Boundary checks that need no GPU: the C-ABI library builds, loads and exports every symbol the header declares;
host-side argument validation and the arena planner (lifetime-based reuse)."""
import ctypes as C
import os
import re

import pytest

from paper_2102_08862_b200 import tracker as T

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "tpc_tracker.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tpc_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = T.load_library()
    names = _declared_functions()
    assert set(names) == set(T.EXPORTS)
    for nm in names:
        assert getattr(lib, nm) is not None
    assert lib.tpc_strerror(0) == b"ok" and b"arena" in lib.tpc_strerror(-2)
    assert lib.tpc_tracker_step_name(0) == b"ingest_radix_sort" and lib.tpc_tracker_step_name(99) is None


def test_arena_bytes_is_host_arithmetic_and_reuses_memory():
    g = T.default_geometry(36, 50485.0)
    n = 150_000_000
    p = T.default_params(max_clusters=n)
    need = T.tpc_tracker_arena_bytes(g, p)
    assert need > 0
    T_cap = n // 10 + 4096
    # sum of all arrays if nothing were reused vs the planned peak
    n_bins = (50485 // 2 + 1) * 36 * 152
    no_reuse = (4 * (n_bins + 1) + 16 * n + 16 * n + 2 * n + 3 * 4 * n + n + 8 * n
                + T_cap * (4 * 160 + 4 * 4 + 28 + 36 + 4 * 5 + 32))
    assert need < 0.85 * no_reuse
    # the floor: what is alive at the same time in the selector (tracklet store + claim + orig + hsr)
    assert need > T_cap * 4 * 160 + 8 * n + 4 * n + 2 * n
    # capacity scaling and host staging only add
    p2 = T.default_params(max_clusters=n)
    p2.host_staging = 1
    assert T.tpc_tracker_arena_bytes(g, p2) >= need
    assert T.tpc_tracker_arena_bytes(g, p, n // 2) < need


def test_invalid_arguments_are_rejected_on_the_host():
    lib = T.load_library()
    g, p = T.default_geometry(), T.default_params(max_clusters=1000)
    bad = T.default_geometry()
    bad.n_rows = 500
    assert T.tpc_tracker_arena_bytes(bad, p) == 0
    long_frame = T.default_geometry(1, 524288.0)            # >= 2^19 time bins: the lookups' fp32 margins no longer hold
    assert T.tpc_tracker_arena_bytes(long_frame, p) == 0
    assert T.tpc_tracker_arena_bytes(T.default_geometry(1, 524287.0), p) > 0
    badp = T.default_params(max_clusters=1000)
    badp.sin_phi_max = 1.5
    assert T.tpc_tracker_arena_bytes(g, badp) == 0
    h = C.c_void_p()
    assert lib.tpc_tracker_create(C.byref(bad), C.byref(p), C.byref(h)) == T.TPC_EINVAL
    assert lib.tpc_tracker_create(C.byref(g), C.byref(p), C.byref(h)) == T.TPC_ENOMEM     # no arena given
    assert lib.tpc_tracker_create(C.byref(g), C.byref(p), None) == T.TPC_EINVAL
    assert lib.tpc_tracker_destroy(None) == T.TPC_EINVAL
    assert lib.tpc_track_timeframe(None, None, 0, None, None) == T.TPC_EINVAL


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        T.Tracker(T.default_geometry(), T.default_params(max_clusters=10))
