"""Pins of the C8 oracle (oracle/tpc_oracle.cpp::orc_refit_chains: one Kalman pass over the hits of a chain of track
pieces linked by C7, with a rotation of state and covariance at every sector boundary).

The paper prints nothing for this step (PAPER.md L23 / L25 only name "full TPC tracking"), so the pins are what the
mathematics and the generator's truth fix: F-J the rotation's covariance factor against the numerical derivative, F-H
noise-free helices (curvature, position and the time re-referencing come out exact), F-N on noisy data the chain fit
resolves q/pT several times better than the innermost piece alone and its variance shrinks, F-I bookkeeping.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle
from oracle import merge as M
from paper_2102_08862_b200 import gen

import merge_eval as ME

_cache = {}


def _refit(cid, seed, **kw):
    key = (cid, seed, tuple(sorted(kw.items())))
    if key not in _cache:
        c = gen.preset(cid, seed)
        for k, v in kw.items():
            setattr(c, k, v)
        tf = gen.generate(c)
        g = oracle.default_geometry(36, tf.max_time_bin)
        p = oracle.default_params(max(c.sigma_y_cm, 0.08), max(c.sigma_z_cm, 0.12))
        res = oracle.track(g, p, tf.row, tf.pad, tf.time)
        mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
        out = oracle.refit_chains(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev)
        _cache[key] = (tf, res, mr, out)
    return _cache[key]


def _truth_k(tf, res):
    keys = ME.track_truth_keys(tf, res.tr_hit_offset, res.tr_n_hits, res.tr_hit_index)
    part = np.where(keys >= 0, keys // (64 * 16), 0)
    outgoing = (keys >= 0) & ((keys % 16) % 2 == 0)          # arc = 2*turn + returning: the tracker sees k = h / pT on outgoing arcs
    return tf.tracks["charge_sense"][part] / tf.tracks["pt"][part], outgoing


@pytest.mark.parametrize("q", [1, -1])
@pytest.mark.parametrize("s0", [-0.6, -0.1, 0.3, 0.7])
def test_FJ_rotation_covariance_factor_is_the_derivative_of_the_rotated_sin_phi(q, s0):
    g, p = oracle.default_geometry(), oracle.default_params()
    cov = [0.04, 0.003, 0.002, 0.01, 0.004, 0.5, 0.09, 0.001, 0.02]
    ok, st, cv = oracle.rotate_with_cov(g, p, [150.0, 20.0, 3.0, s0, 0.4, 1.2], cov, q)
    assert ok
    delta = math.radians(20.0) * q
    f = lambda s: math.sin(math.asin(s) - delta)
    eps = 1e-6
    J = (f(s0 + eps) - f(s0 - eps)) / (2 * eps)
    assert abs(st[3] - f(s0)) < 2e-6
    assert abs(cv[1] / cov[1] - J) < 1e-5 and abs(cv[4] / cov[4] - J) < 1e-5 and abs(cv[2] / cov[2] - J * J) < 2e-5
    for i in (0, 3, 5, 6, 7, 8):                              # yy, yk, kk and the (z, t) block are untouched
        assert cv[i] == np.float32(cov[i])
    # the point itself: rotation about the beam axis
    assert abs(st[0] - (150.0 * math.cos(delta) + 20.0 * math.sin(delta))) < 2e-4
    assert abs(st[1] - (-150.0 * math.sin(delta) + 20.0 * math.cos(delta))) < 2e-4


def test_FJ_rotation_fails_beyond_sin_phi_max_and_keeps_the_state():
    g, p = oracle.default_geometry(), oracle.default_params()
    cov = [1, 0, 0.1, 0, 0, 100, 1, 0, 0.1]
    ok, st, cv = oracle.rotate_with_cov(g, p, [150.0, 20.0, 3.0, 0.9, 0.4, 1.2], cov, -1)      # asin(0.9) + 20 deg > asin(0.95)
    assert not ok
    np.testing.assert_array_equal(st, np.array([150.0, 20.0, 3.0, 0.9, 0.4, 1.2], np.float32))


def test_FH_noise_free_helices_are_refitted_exactly():
    tf, res, mr, (ok, ch, cp, rp, rc) = _refit(1, 4, fixed_tracks=600, sigma_y_cm=0.0, sigma_z_cm=0.0, dropout=0.0, noise_frac=0.0, pt_min=0.15)
    roots = np.nonzero((mr.prev < 0) & (mr.next >= 0))[0]
    assert roots.size > 400 and np.all(ok[roots] == 1) and (cp[roots] == 3).any()
    k_true, outgoing = _truth_k(tf, res)
    sel = roots[outgoing[roots]]
    assert sel.size > 300
    assert np.max(np.abs(rp[sel, 5] - k_true[sel]) / np.abs(k_true[sel])) < 1e-3
    # the state sits on the innermost hit of the innermost piece: y and the re-referenced z reproduce that hit
    n_pads = np.floor(2.0 * (85.0 + 1.07 * np.arange(152)) * math.tan(math.radians(10.0)) / 0.5)
    for i in sel[:200]:
        h = res.tr_hit_index[res.tr_hit_offset[i]]
        r = int(tf.row[h]) % 152
        assert abs(rp[i, 0] - (85.0 + 1.07 * r)) < 1e-4
        assert abs(rp[i, 1] - (tf.pad[h] - 0.5 * (n_pads[r] - 1)) * 0.5) < 2e-3
        assert abs(rp[i, 2] - (tf.time[h] - rp[i, 6]) * 0.516) < 2e-3
        assert rp[i, 6] == res.tr_par[i, 6]


@pytest.mark.parametrize("seed", [1, 2])
def test_FN_chain_fit_resolves_curvature_better_than_the_innermost_piece(seed):
    tf, res, mr, (ok, ch, cp, rp, rc) = _refit(1, seed)
    roots = np.nonzero((mr.prev < 0) & (mr.next >= 0))[0]
    assert roots.size > 2500
    assert (ok[roots] == -1).mean() < 0.02 and np.all(ok[roots] != 0)
    k_true, outgoing = _truth_k(tf, res)
    sel = roots[(ok[roots] == 1) & outgoing[roots]]
    err_piece = np.median(np.abs(res.tr_par[sel, 5] - k_true[sel]))
    err_chain = np.median(np.abs(rp[sel, 5] - k_true[sel]))
    assert err_chain < 0.25 * err_piece, (err_chain, err_piece)
    assert np.mean(rc[sel, 5] < res.tr_cov[sel, 5]) > 0.99                    # kk variance shrinks
    assert np.all(rc[sel][:, [0, 2, 5, 6, 8]] > 0)                            # diagonal stays positive
    pull = (rp[sel, 5] - k_true[sel]) / np.sqrt(rc[sel, 5])
    assert 0.5 < np.std(pull[np.abs(pull) < 10]) < 2.0                        # the quoted variance is the scatter


def test_FI_bookkeeping():
    tf, res, mr, (ok, ch, cp, rp, rc) = _refit(1, 1)
    n = len(ok)
    roots = (mr.prev < 0) & (mr.next >= 0)
    assert np.all(ok[~roots] == 0)
    np.testing.assert_array_equal(rp[~roots], res.tr_par[~roots])             # not a chain root: parameters passed through
    assert np.all(rc[~roots] == 0)
    np.testing.assert_array_equal(ch[~roots], res.tr_n_hits[~roots])
    hits_by_root = np.bincount(mr.root, weights=res.tr_n_hits, minlength=n).astype(np.int64)
    pieces_by_root = np.bincount(mr.root, minlength=n)
    np.testing.assert_array_equal(ch[roots], hits_by_root[roots])
    np.testing.assert_array_equal(cp[roots], pieces_by_root[roots])
    failed = ok == -1
    np.testing.assert_array_equal(rp[failed], res.tr_par[failed])             # a failed chain keeps the root's parameters
