"""Pins of the synthetic generator (inputs only): helix closed forms, determinism, the configs' sizes (G2)."""
import math

import numpy as np

from helpers import N_ROWS, n_pads, row_x
from paper_2102_08862_b200 import gen


def _clean(cid=0, seed=3, **kw):
    c = gen.preset(cid, seed)
    c.sigma_y_cm = c.sigma_z_cm = c.dropout = c.noise_frac = 0.0
    for k, v in kw.items():
        setattr(c, k, v)
    return gen.generate(c)


def test_G2_crossings_lie_on_the_helix():
    """Every noise-free cluster satisfies sin(phi_local)(x_r) = sin(psi0) + h x_r / R, the circle equation and
    z = z_v + R theta sinh(eta) (SURVEY.md §8(d) closed form; BASELINE.json L7: R = 666.7 pT cm)."""
    tf = _clean(1, 5, fixed_tracks=200)
    sr = tf.row.astype(np.int64)
    sector, r = sr // N_ROWS, sr % N_ROWS
    x = row_x(r)
    y = (tf.pad.astype(np.float64) - 0.5 * (n_pads(r) - 1)) * 0.5
    tr = tf.tracks[tf.truth_track]
    R = 666.7 * tr["pt"]
    h = tr["charge_sense"].astype(np.float64)
    alpha = np.radians(20.0 * (sector % 18) + 10.0)
    psi0 = tr["phi0"] - alpha
    xc, yc = -(R / h) * np.sin(psi0), (R / h) * np.cos(psi0)
    assert np.max(np.abs(np.hypot(x - xc, y - yc) - R) / R) < 1e-6
    v = np.sin(psi0) + h * x / R
    assert np.all(np.abs(v) <= 1.0)
    ret = (tf.truth_arc % 2).astype(bool)
    cpsi = np.where(ret, -1.0, 1.0) * np.sqrt(1 - v * v)
    np.testing.assert_allclose(y, (R / h) * (np.cos(psi0) - cpsi), atol=2e-5)
    theta = np.mod(h * (np.arctan2(v, cpsi) - psi0), 2 * np.pi) + 2 * np.pi * (tf.truth_arc // 2)
    z = tr["z_v"] + R * theta * np.sinh(tr["eta"])
    np.testing.assert_allclose(tf.time.astype(np.float64) * 0.516, 250.0 - np.abs(z), atol=3e-5)
    assert np.array_equal(sector >= 18, z < 0)


def test_generator_is_deterministic_and_shuffled():
    a = gen.generate(gen.preset(0, 1))
    b = gen.generate(gen.preset(0, 1))
    c = gen.generate(gen.preset(0, 2))
    for name in ("row", "pad", "time", "charge", "truth_track", "truth_arc"):
        assert np.array_equal(getattr(a, name), getattr(b, name))
    assert a.n != c.n or not np.array_equal(a.pad, c.pad)
    cfg = gen.preset(0, 1); cfg.n_threads = 1
    d = gen.generate(cfg)
    assert np.array_equal(a.time, d.time)                  # independent of the thread count
    cfg = gen.preset(0, 1); cfg.shuffle = 0
    u = gen.generate(cfg)
    assert u.n == a.n and not np.array_equal(u.time, a.time)
    assert np.array_equal(np.sort(u.time), np.sort(a.time))  # the shuffle is a permutation
    # noise fraction and label conventions
    assert (a.truth_track < 0).sum() == round(0.05 * a.n_real)
    assert a.row.min() >= 0 and a.row.max() < N_ROWS and np.all(a.row == np.floor(a.row))


def test_config_sizes():
    """configs[0] / [1] of BASELINE.json: 300 resp. 4000 tracks, one collision, time within one drift length."""
    a, b = gen.generate(gen.preset(0, 1)), gen.generate(gen.preset(1, 1))
    assert len(a.tracks) == 300 and len(b.tracks) == 4000 and a.n_collisions == b.n_collisions == 1
    assert 5e3 < a.n < 1e5 and 3e5 < b.n < 3e6
    assert b.row.max() < 36 * N_ROWS and a.time.max() <= a.max_time_bin and b.time.max() <= b.max_time_bin
    c = gen.generate(gen.preset(2, 1, frame_us=100.0))
    assert c.n_collisions >= 1 and c.time.max() <= c.max_time_bin
    pt = b.tracks["pt"]
    assert pt.min() >= 0.1 and pt.max() <= 20.0 and abs(np.mean(pt) - 0.6) < 0.05
    assert np.abs(b.tracks["eta"]).max() <= 0.9
