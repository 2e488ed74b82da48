"""Pins of the C11 oracle (oracle/tpc_oracle.cpp::orc_compress_tracks: track-based hit rejection + track-model residual
coding).  PAPER.md L23 names the two operations and prints nothing else, so the pins are what the
definition fixes: Q-R decode(encode(hits)) = hits within half a step, Q-C the coder restated step by step with the (separately
pinned) transport / update hooks, Q-J the rejection rule, Q-H noise-free helices code to ~zero symbols, Q-E the entropy of the
symbols against the raw coordinates at the same quantisation."""
import numpy as np
import pytest

import oracle
from helpers import N_ROWS, n_pads
from paper_2102_08862_b200 import gen

_cache = {}


def _tracked(cid, seed, **kw):
    key = (cid, seed, tuple(sorted(kw.items())))
    if key not in _cache:
        c = gen.preset(cid, seed)
        for k, v in kw.items():
            setattr(c, k, v)
        tf = gen.generate(c)
        g = oracle.default_geometry(c.n_sectors, tf.max_time_bin)
        p = oracle.default_params(max(c.sigma_y_cm, 0.08), max(c.sigma_z_cm, 0.12))
        res = oracle.track(g, p, tf.row, tf.pad, tf.time)
        _cache[key] = (tf, g, p, res)
    return _cache[key]


def _hit_truth(tf, res):
    hi = res.tr_hit_index
    r = (tf.row[hi].astype(np.int64) % N_ROWS)
    cr = (0.5 * (n_pads(np.arange(N_ROWS)) - 1)).astype(np.float32)
    y = (tf.pad[hi] - cr[r]) * np.float32(0.5)
    z = (tf.time[hi] - np.repeat(res.tr_par[:, 6], res.tr_n_hits)) * np.float32(0.516)
    return r.astype(np.uint8), y, z


def _entropy(x):
    _, c = np.unique(x, return_counts=True)
    pr = c / c.sum()
    return float(-(pr * np.log2(pr)).sum())


@pytest.mark.parametrize("step,step_z", [(0.025, 0.025), (0.01, 0.04), (0.1, 0.03)])
def test_QR_decoder_reproduces_every_hit_within_half_a_step(step, step_z):
    tf, g, p, res = _tracked(1, 1)
    rej, ok, qy, qz = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, step_y=step, step_z=step_z)
    hr, y, z = _hit_truth(tf, res)
    yd, zd = oracle.decompress_tracks(g, p, res, hr, ok, qy, qz, step_y=step, step_z=step_z)
    keep = np.repeat(ok == 1, res.tr_n_hits)
    assert keep.sum() > 6e5 and (ok == 0).sum() < 0.005 * len(ok)
    assert np.max(np.abs(yd - y)[keep]) <= 0.5 * step * 1.001 + 1e-5 and np.max(np.abs(zd - z)[keep]) <= 0.5 * step_z * 1.001 + 1e-5
    # the symbols scale with their OWN step: spread (in cm) of the coded residuals is the same whatever the steps
    assert 0.05 < qy[keep].std() * step < 0.2 and 0.08 < qz[keep].std() * step_z < 0.3
    assert np.all(np.isnan(yd[~keep]))
    assert np.abs(qy).max() < 32767 and np.abs(qz).max() < 32767


def test_QC_coder_restated_with_the_transport_and_update_hooks():
    """The closed loop, one track at a time in Python: transport -> residual -> rintf(residual / step) -> update with the
    RECONSTRUCTED hit.  Symbols identical for every hit of 40 tracks."""
    tf, g, p, res = _tracked(0, 2)
    step = np.float32(0.025)
    rej, ok, qy, qz = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res)
    hr, y, z = _hit_truth(tf, res)
    x_r, _, _, k = oracle.tables(g, p)
    f = np.float32
    done = 0
    for t in range(len(res.tr_seed)):
        if ok[t] != 1:
            continue
        st, cv = res.tr_par[t, :6].copy(), res.tr_cov[t].copy()
        o, n = int(res.tr_hit_offset[t]), int(res.tr_n_hits[t])
        for j in range(o, o + n):
            good, st, cv = oracle.transport(p, st, cv, float(x_r[hr[j]]))
            assert good
            ry, rz = f(y[j] - st[1]), f(z[j] - st[2])
            iy, iz = int(np.rint(f(ry / step))), int(np.rint(f(rz / step)))
            assert (iy, iz) == (int(qy[j]), int(qz[j])), (t, j)
            yq, zq = f(st[1] + f(f(iy) * step)), f(st[2] + f(f(iz) * step))
            st, cv = oracle.update(st, cv, float(yq), float(zq), float(k["ry"]), float(k["rz"]))
        done += 1
        if done == 40:
            break
    assert done == 40


def test_QJ_rejection_rule():
    tf, g, p, res = _tracked(1, 2)
    cut = 1.0 / 0.2
    rej, ok, qy, qz = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, reject_qpt=cut)
    low = np.abs(res.tr_par[:, 5]) > np.float32(cut)
    assert 200 < low.sum() < 0.5 * len(low)
    np.testing.assert_array_equal(ok == -1, low)
    expect = np.zeros(tf.n, np.uint8)
    expect[res.tr_hit_index[np.repeat(low, res.tr_n_hits)]] = 1
    np.testing.assert_array_equal(rej, expect)
    assert np.all(qy[np.repeat(low, res.tr_n_hits)] == 0)
    owned = np.zeros(tf.n, bool); owned[res.tr_hit_index] = True
    assert not rej[~owned].any()                                   # hits no track owns are kept
    none = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, reject_qpt=1e9)
    assert none[0].sum() == 0 and (none[1] == -1).sum() == 0
    # the bound is strict: a track with |q/pT| exactly on the cut is kept, one float below the cut it is rejected
    k_abs = np.abs(res.tr_par[:, 5])
    i = int(np.argsort(k_abs)[len(k_abs) // 2])
    on = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, reject_qpt=float(k_abs[i]))
    below = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, reject_qpt=float(np.nextafter(k_abs[i], np.float32(0))))
    assert on[1][i] != -1 and below[1][i] == -1


def test_QH_noise_free_helices_code_to_almost_nothing():
    tf, g, p, res = _tracked(1, 4, fixed_tracks=400, sigma_y_cm=0.0, sigma_z_cm=0.0, dropout=0.0, noise_frac=0.0, pt_min=0.3)
    rej, ok, qy, qz = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res)
    keep = np.repeat(ok == 1, res.tr_n_hits)
    assert keep.sum() > 2e4
    assert np.mean(np.abs(qy[keep]) <= 1) > 0.99 and np.mean(np.abs(qz[keep]) <= 1) > 0.99      # the model IS the data
    assert _entropy(qy[keep]) < 1.5 and _entropy(qz[keep]) < 1.5


@pytest.mark.parametrize("cid,seed", [(1, 1), (0, 3)])
def test_QE_entropy_of_the_symbols_against_the_raw_coordinates(cid, seed):
    tf, g, p, res = _tracked(cid, seed)
    step = 0.025
    rej, ok, qy, qz = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res)
    keep = np.repeat(ok == 1, res.tr_n_hits)
    hi = res.tr_hit_index[keep]
    raw_y = np.rint(tf.pad[hi].astype(np.float64) * 0.5 / step).astype(np.int64)          # the same coordinates, same quantisation
    raw_z = np.rint(tf.time[hi].astype(np.float64) * 0.516 / step).astype(np.int64)
    h_res, h_raw = _entropy(qy[keep]) + _entropy(qz[keep]), _entropy(raw_y) + _entropy(raw_z)
    assert h_res < 0.45 * h_raw, (h_res, h_raw)
    # the symbol spread is the prediction error in steps: a few steps for sigma_y 0.08 / sigma_z 0.12 at a 0.025 cm step
    assert 2.0 < qy[keep].std() < 6.0 and 3.0 < qz[keep].std() < 9.0
    # halving the step costs about one bit per coordinate
    _, ok2, qy2, qz2 = oracle.compress_tracks(g, p, tf.row, tf.pad, tf.time, res, step_y=step / 2, step_z=step / 2)
    k2 = np.repeat(ok2 == 1, res.tr_n_hits)
    assert 1.5 < _entropy(qy2[k2]) + _entropy(qz2[k2]) - h_res < 2.5
