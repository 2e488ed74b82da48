"""tpc_find_clusters_static: the cluster finder (C0) for callers that must not allocate -- no tracker handle, no arena, its
scratch a fixed array inside the library image (include/tpc_tracker.h).  Checked against the existing path
(tpc_find_clusters with an arena) on the same inputs, bit for bit like tests/test_cluster_gpu.py, on two calls in a row whose
inputs differ in size (the second call finds the first call's contents in the shared scratch).

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`.
"""
from __future__ import annotations

import numpy as np
import pytest

from paper_2102_08862_b200 import gen

pytestmark = pytest.mark.gpu


def _digits(cid, seed, frame_us=None):
    c = gen.preset(cid, seed, frame_us)
    tf = gen.generate(c, want_truth=False)
    return tf, gen.digitize(tf.row, tf.pad, tf.time, tf.charge, c.n_sectors, tf.max_time_bin)


def _existing_path(T, torch, dev_digits, n, n_sectors, max_time_bin):
    trk = T.Tracker(T.default_geometry(n_sectors, max_time_bin), T.default_params(max_clusters=max(n, 1)))
    out = trk.tpc_find_clusters(*dev_digits, n=n)
    torch.cuda.synchronize()
    k = int(out[4][0])
    res = [out[i][:k].cpu().numpy() for i in range(4)] + [k, int(out[5][0])]
    trk.close()
    return res


def test_static_scratch_cluster_finder_equals_the_arena_path_on_two_calls_in_a_row():
    import torch
    from paper_2102_08862_b200 import tracker as T
    limit = T.tpc_find_clusters_static_max_digits()
    assert limit == 1 << 20
    tf_a, d_a = _digits(1, 1)                     # full TPC: 3.3e6 samples, cut to the limit (a prefix of a sorted input is sorted)
    tf_b, d_b = _digits(0, 5)                     # one sector, 7e4 samples: ends in the middle of a tile
    assert d_a.n > limit and 10_000 < d_b.n < limit and d_b.n % 2048 != 0
    dev = torch.device("cuda:0")
    cases = []
    for tf, d, n, n_sec in ((tf_a, d_a, limit, 36), (tf_b, d_b, d_b.n, 1)):
        t = [torch.from_numpy(np.ascontiguousarray(a[:n])).to(dev) for a in (d.row, d.pad, d.time, d.adc)]
        cases.append((t, n, _existing_path(T, torch, t, n, n_sec, tf.max_time_bin)))
    # outputs are the caller's; allocate them BEFORE the calls under test
    cap = limit
    out = (torch.empty(cap, dtype=torch.float32, device=dev), torch.empty(cap, dtype=torch.float32, device=dev),
           torch.empty(cap, dtype=torch.float32, device=dev), torch.empty(cap, dtype=torch.float32, device=dev),
           torch.empty(1, dtype=torch.int64, device=dev), torch.empty(1, dtype=torch.int32, device=dev))
    T.tpc_find_clusters_static_setup()
    torch.cuda.synchronize()
    allocated = torch.cuda.memory_allocated(dev)
    for rep in range(2):                           # A, B, A, B: every call after the first finds another call's scratch contents
        for t, n, ref in cases:
            for o in out[:4]:
                o.fill_(-1.0)
            T.tpc_find_clusters_static(*t, out=out, n=n)
            torch.cuda.synchronize()
            k = int(out[4][0])
            assert k == ref[4] and int(out[5][0]) == ref[5] == 0 and k > 0.1 * n / 5.5
            for i, nm in enumerate(("row", "pad", "time", "charge")):
                assert np.array_equal(out[i][:k].cpu().numpy().view(np.uint32), ref[i].view(np.uint32)), (nm, rep, n)
            assert float(out[1][k]) == -1.0 if k < cap else True       # nothing written behind the clusters
    assert torch.cuda.memory_allocated(dev) == allocated
    # sizes beyond the built-in scratch are refused with a clear error, nothing enqueued; n = 0 is fine
    big = [torch.zeros(limit + 1, dtype=dt, device=dev) for dt in (torch.int32, torch.int32, torch.int32, torch.float32)]
    with pytest.raises(T.TpcError) as e:
        T.tpc_find_clusters_static(*big, out=out, n=limit + 1)
    assert e.value.code == T.TPC_ENOMEM
    T.tpc_find_clusters_static(*big, out=out, n=0)
    torch.cuda.synchronize()
    assert int(out[4][0]) == 0 and int(out[5][0]) == 0
    # capacity smaller than the result: status 1, the count reported, a valid prefix written (as the arena path)
    t, n, ref = cases[1]
    small = tuple(torch.empty(100, dtype=torch.float32, device=dev) for _ in range(4)) + (out[4], out[5])
    T.tpc_find_clusters_static(*t, out=small, n=n)
    torch.cuda.synchronize()
    assert int(out[5][0]) == 1 and int(out[4][0]) == ref[4] and np.array_equal(small[1].cpu().numpy(), ref[1][:100])
