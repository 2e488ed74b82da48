"""Runs the CUDA path and the oracle on the same clusters and compares them (used by the -m gpu tests and smoke()).

Bar (BASELINE.json L5): neighbour links, start hits and tracklet-to-hit assignments bit-exact; fitted y, z within
1e-3 cm; q/pT within 1e-4 relative.  Both sides take every decision in fp32 with the same operation order, so the
fits are expected to be bit-identical too; the tolerances are what is asserted, bit-identity is reported.
"""
from __future__ import annotations

import numpy as np

Y_Z_TOL_CM = 1e-3
QPT_REL_TOL = 1e-4


def run_gpu(row, pad, time, n_sectors, max_time_bin, sigma_y=0.08, sigma_z=0.12, taps=True, **param_overrides):
    import torch
    from paper_2102_08862_b200 import tracker as T
    n = int(len(row))
    g = T.default_geometry(n_sectors, max_time_bin)
    p = T.default_params(sigma_y, sigma_z, max_clusters=max(n, 1))
    for k, v in param_overrides.items():
        setattr(p, k, v)
    trk = T.Tracker(g, p)
    dev = trk.device
    d = [torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(dev) for a in (row, pad, time)]
    out = trk.tpc_track_timeframe(*d, n=n, taps=taps)
    torch.cuda.synchronize()
    res = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.__dict__.items()}
    res["launches"] = trk.last_launches()
    res["work"] = trk.work_counters()
    trk.close()
    return res


def run_oracle(row, pad, time, n_sectors, max_time_bin, sigma_y=0.08, sigma_z=0.12, **param_overrides):
    import oracle
    g = oracle.default_geometry(n_sectors, max_time_bin)
    p = oracle.default_params(sigma_y, sigma_z)
    for k, v in param_overrides.items():
        if k != "follower":                   # a knob of the CUDA path only (which follower kernel runs)
            setattr(p, k, v)
    return oracle.track(g, p, row, pad, time)


def compare(gpu: dict, orc, n_rows: int = 152) -> dict:
    """Asserts the parity bar; returns a small report."""
    rep = {}
    # links and start hits: bit-exact, by original index
    np.testing.assert_array_equal(gpu["link_up"], orc.link_up, err_msg="link_up")
    np.testing.assert_array_equal(gpu["link_down"], orc.link_down, err_msg="link_down")
    np.testing.assert_array_equal(gpu["is_start_hit"], orc.is_start_hit, err_msg="is_start_hit")
    # tracklets: join on the seed (= tracklet id)
    nt = int(gpu["n_tracklets"][0])
    assert nt == len(orc.tl_seed), (nt, len(orc.tl_seed))
    g_seed = gpu["tracklet_seed"][:nt]
    order = np.argsort(g_seed, kind="stable")
    np.testing.assert_array_equal(g_seed[order], orc.tl_seed, err_msg="tracklet seeds")   # oracle: ascending seed
    np.testing.assert_array_equal(gpu["tracklet_n_hits"][:nt][order], orc.tl_n_hits, err_msg="tracklet n_hits")
    np.testing.assert_array_equal(gpu["tracklet_row_hit"][:nt][order], orc.tl_row_hit, err_msg="tracklet row->hit")
    gp = gpu["tracklet_par"][:nt][order]
    rep["tracklet_par_bit_identical"] = bool(np.array_equal(gp, orc.tl_par))
    _check_par(gp, orc.tl_par, "tracklet")
    # tracks: join on seed_hit
    k = int(gpu["n_tracks"][0])
    assert int(gpu["status"][0]) & 7 == 0, f"overflow status {int(gpu['status'][0])}"
    assert k == len(orc.tr_seed), (k, len(orc.tr_seed))
    assert int(gpu["n_track_hits"][0]) == len(orc.tr_hit_index)
    gs = gpu["seed_hit"][:k]
    go = np.argsort(gs, kind="stable")
    oo = np.argsort(orc.tr_seed, kind="stable")
    np.testing.assert_array_equal(gs[go], orc.tr_seed[oo], err_msg="track seeds")
    for name, ref in (("sector", orc.tr_sector), ("first_row", orc.tr_first_row), ("last_row", orc.tr_last_row),
                      ("n_hits", orc.tr_n_hits)):
        np.testing.assert_array_equal(gpu[name][:k][go], ref[oo], err_msg=f"track {name}")
    g_off, g_n = gpu["hit_offset"][:k][go], gpu["n_hits"][:k][go]
    for a in range(k):
        gh = gpu["hit_index"][g_off[a]:g_off[a] + g_n[a]]
        np.testing.assert_array_equal(gh, orc.track_hits(int(oo[a])), err_msg=f"hits of track seed {gs[go][a]}")
    gpar = np.stack([gpu[nm][:k][go] for nm in ("x", "y", "z_rel", "sin_phi", "dzds", "q_pt", "time_ref")], 1)
    rep["track_par_bit_identical"] = bool(np.array_equal(gpar, orc.tr_par[oo]))
    rep["track_cov_bit_identical"] = bool(np.array_equal(gpu["cov9"][:k][go], orc.tr_cov[oo]))
    _check_par(gpar, orc.tr_par[oo], "track")
    # every hit in at most one track
    hi = gpu["hit_index"][:int(gpu["n_track_hits"][0])]
    assert np.unique(hi).size == hi.size
    rep.update(n_tracklets=nt, n_tracks=k, n_track_hits=int(hi.size), n_links=int((orc.link_up >= 0).sum()),
               n_start_hits=int(orc.is_start_hit.sum()))
    return rep


def _check_par(g, o, what):
    if g.shape[0] == 0:
        return
    assert np.all(np.isfinite(g)), f"{what}: non-finite fitted parameter"
    assert np.max(np.abs(g[:, 0] - o[:, 0])) == 0, f"{what} x"
    assert np.max(np.abs(g[:, 1] - o[:, 1])) <= Y_Z_TOL_CM, f"{what} y"
    assert np.max(np.abs(g[:, 2] - o[:, 2])) <= Y_Z_TOL_CM, f"{what} z"
    assert np.max(np.abs(g[:, 3] - o[:, 3])) <= 1e-4, f"{what} sin_phi"
    assert np.max(np.abs(g[:, 4] - o[:, 4])) <= 1e-4, f"{what} dzds"
    den = np.maximum(np.abs(o[:, 5]), 1e-3)
    assert np.max(np.abs(g[:, 5] - o[:, 5]) / den) <= QPT_REL_TOL, f"{what} q/pT"
    assert np.array_equal(g[:, 6], o[:, 6]), f"{what} time_ref"


def run_oracle_per_sector(row, pad, time, n_sectors, max_time_bin, sigma_y=0.08, sigma_z=0.12, threads=None, n_rows=152):
    """The unchanged oracle, one call per sector from a thread pool (ctypes releases the GIL), results mapped back to
    whole-frame cluster indices.  Sectors are independent (reading A16) and a sub-frame keeps the cluster order, so
    every original-index tie-break and tracklet id maps through the selection.  Returns a dict of whole-frame arrays;
    per-sector results are reduced at once (the tracklets' row->hit tables are dropped: 10 GB for a 10 ms frame)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    import oracle
    n = int(len(row))
    sec = (row.astype(np.int32) // n_rows)
    order = np.argsort(sec, kind="stable")                      # ascending cluster index inside a sector
    bounds = np.searchsorted(sec[order], np.arange(n_sectors + 1))
    g1 = oracle.default_geometry(1, max_time_bin)
    p = oracle.default_params(sigma_y, sigma_z)
    oracle.lib()
    up = np.full(n, -1, np.int32); down = np.full(n, -1, np.int32); start = np.zeros(n, np.uint8)

    def one(s):
        sel = order[bounds[s]:bounds[s + 1]]
        if sel.size == 0:
            return None
        r = oracle.track(g1, p, row[sel] - np.float32(s * n_rows), pad[sel], time[sel])
        sel32 = sel.astype(np.int32)
        up[sel] = np.where(r.link_up >= 0, sel32[np.maximum(r.link_up, 0)], -1)
        down[sel] = np.where(r.link_down >= 0, sel32[np.maximum(r.link_down, 0)], -1)
        start[sel] = r.is_start_hit
        return dict(tl_seed=sel32[r.tl_seed], tl_n_hits=r.tl_n_hits, tl_par=r.tl_par,
                    tr_seed=sel32[r.tr_seed], tr_sector=np.full(len(r.tr_seed), s, np.int32), tr_first_row=r.tr_first_row,
                    tr_last_row=r.tr_last_row, tr_n_hits=r.tr_n_hits, tr_par=r.tr_par, tr_cov=r.tr_cov,
                    tr_hit_index=sel32[r.tr_hit_index])

    threads = threads or max(1, min(n_sectors, os.cpu_count() or 1))
    with ThreadPoolExecutor(threads) as ex:
        parts = [q for q in ex.map(one, range(n_sectors)) if q is not None]
    res = {k: np.concatenate([q[k] for q in parts]) for k in parts[0]} if parts else {}
    res.update(link_up=up, link_down=down, is_start_hit=start)
    return res


def _ragged_gather(values, offsets, counts):
    """Concatenation of values[offsets[i] : offsets[i] + counts[i]] over i, vectorised."""
    counts = counts.astype(np.int64)
    total = int(counts.sum())
    starts = np.concatenate([[0], np.cumsum(counts[:-1])]) if counts.size else np.zeros(0, np.int64)
    idx = np.arange(total, dtype=np.int64) - np.repeat(starts, counts) + np.repeat(offsets.astype(np.int64), counts)
    return values[idx]


def compare_whole_frame(gpu: dict, orc: dict) -> dict:
    """Bit-for-bit comparison of a whole frame (arrays by original cluster index / joined on the seed)."""
    np.testing.assert_array_equal(gpu["link_up"], orc["link_up"], err_msg="link_up")
    np.testing.assert_array_equal(gpu["link_down"], orc["link_down"], err_msg="link_down")
    np.testing.assert_array_equal(gpu["is_start_hit"], orc["is_start_hit"], err_msg="is_start_hit")
    nt = int(gpu["n_tracklets"][0])
    assert nt == len(orc["tl_seed"]), (nt, len(orc["tl_seed"]))
    go, oo = np.argsort(gpu["tracklet_seed"][:nt], kind="stable"), np.argsort(orc["tl_seed"], kind="stable")
    np.testing.assert_array_equal(gpu["tracklet_seed"][:nt][go], orc["tl_seed"][oo], err_msg="tracklet seeds")
    np.testing.assert_array_equal(gpu["tracklet_n_hits"][:nt][go], orc["tl_n_hits"][oo], err_msg="tracklet n_hits")
    assert np.array_equal(gpu["tracklet_par"][:nt][go].view(np.uint32), orc["tl_par"][oo].view(np.uint32)), "tracklet parameters"
    k = int(gpu["n_tracks"][0])
    assert k == len(orc["tr_seed"]), (k, len(orc["tr_seed"]))
    go, oo = np.argsort(gpu["seed_hit"][:k], kind="stable"), np.argsort(orc["tr_seed"], kind="stable")
    np.testing.assert_array_equal(gpu["seed_hit"][:k][go], orc["tr_seed"][oo], err_msg="track seeds")
    for name, ref in (("sector", "tr_sector"), ("first_row", "tr_first_row"), ("last_row", "tr_last_row"), ("n_hits", "tr_n_hits")):
        np.testing.assert_array_equal(gpu[name][:k][go], orc[ref][oo], err_msg=f"track {name}")
    o_off = np.concatenate([[0], np.cumsum(orc["tr_n_hits"][:-1], dtype=np.int64)]) if k else np.zeros(0, np.int64)
    gh = _ragged_gather(gpu["hit_index"], gpu["hit_offset"][:k][go], gpu["n_hits"][:k][go])
    oh = _ragged_gather(orc["tr_hit_index"], o_off[oo], orc["tr_n_hits"][oo])
    np.testing.assert_array_equal(gh, oh, err_msg="track hit lists")
    gpar = np.stack([gpu[nm][:k][go] for nm in ("x", "y", "z_rel", "sin_phi", "dzds", "q_pt", "time_ref")], 1)
    assert np.array_equal(gpar.view(np.uint32), orc["tr_par"][oo].view(np.uint32)), "track parameters"
    assert np.array_equal(gpu["cov9"][:k][go].view(np.uint32), orc["tr_cov"][oo].view(np.uint32)), "track covariance"
    return dict(n_tracks_compared=k, n_tracks_oracle=len(orc["tr_seed"]), n_track_hits_compared=int(gh.size),
                n_tracklets_compared=nt, n_links_compared=int(gpu["link_up"].size))
