"""tpc_track_timeframe only enqueues work (no allocation, no synchronisation: include/tpc_tracker.h), so a caller can capture
it in a CUDA graph and replay it -- what pays on the small configurations, whose ~46 launches per frame cost more than their
kernels.  The replayed graph must give the eager call's result bit for bit, also after the input buffers were refilled with
another frame of the same size."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2102_08862_b200 import gen

pytestmark = pytest.mark.gpu


def _snapshot(out):
    k, nh = int(out.n_tracks[0]), int(out.n_track_hits[0])
    f = ("seed_hit", "sector", "first_row", "last_row", "n_hits", "hit_offset", "x", "y", "z_rel", "time_ref", "sin_phi", "dzds", "q_pt", "cov9")
    return k, nh, int(out.status[0]), [getattr(out, a)[:k].cpu().numpy().copy() for a in f], out.hit_index[:nh].cpu().numpy().copy()


def _same(a, b):
    assert a[0] == b[0] and a[1] == b[1] and a[2] == b[2]
    for x, y in zip(a[3], b[3]):
        assert np.array_equal(x.view(np.uint8), y.view(np.uint8))
    assert np.array_equal(a[4], b[4])


@pytest.mark.parametrize("cid", [0, 1])
def test_a_captured_frame_replays_bit_identically_also_on_new_input(cid):
    import torch
    from paper_2102_08862_b200 import tracker as T
    cfg_a, cfg_b = gen.preset(cid, 1), gen.preset(cid, 2)
    tf_a, tf_b = gen.generate(cfg_a, want_truth=False), gen.generate(cfg_b, want_truth=False)
    n = min(tf_a.n, tf_b.n)                                    # a graph is captured for ONE n (grid sizes are launch parameters)
    trk = T.Tracker(T.default_geometry(cfg_a.n_sectors, max(tf_a.max_time_bin, tf_b.max_time_bin)),
                    T.default_params(cfg_a.sigma_y_cm, cfg_a.sigma_z_cm, max_clusters=n))
    dev = trk.device
    buf = [torch.empty(n, dtype=torch.float32, device=dev) for _ in range(3)]
    load = lambda tf: [b.copy_(torch.from_numpy(np.ascontiguousarray(a[:n]))) for b, a in zip(buf, (tf.row, tf.pad, tf.time))]
    outs = trk.alloc_outputs(n)
    load(tf_a)
    eager_a = _snapshot(trk.tpc_track_timeframe(*buf, n=n, outputs=outs))
    load(tf_b)
    eager_b = _snapshot(trk.tpc_track_timeframe(*buf, n=n, outputs=outs))
    assert eager_a[0] > 50 and eager_a[1] != eager_b[1]
    torch.cuda.synchronize()
    s = torch.cuda.Stream(device=dev)
    graph = torch.cuda.CUDAGraph()
    load(tf_a)
    torch.cuda.synchronize()
    with torch.cuda.graph(graph, stream=s):
        trk.tpc_track_timeframe(*buf, n=n, outputs=outs, stream=torch.cuda.current_stream(dev))
    for tf, ref in ((tf_a, eager_a), (tf_b, eager_b), (tf_a, eager_a)):
        load(tf)
        for o in (outs[0].n_tracks, outs[0].n_track_hits):
            o.zero_()
        graph.replay()
        torch.cuda.synchronize()
        _same(_snapshot(outs[0]), ref)
    trk.close()
