"""Pins of the C7 oracle (oracle/tpc_merge_oracle.cpp: sector-boundary merging of the per-sector tracks).

The paper prints no worked example of the merger (PAPER.md L23/L25 only name "full TPC tracking"), so the pins are
what geometry and the generator's truth fix: M-R the rotation against the double-precision helix in GLOBAL
coordinates, M-T the state-only transport against the (separately pinned, K1) full transport, M-H noise-free helices
that cross sector boundaries, M-I invariants, M-P independence of the input order, M-E efficiency / purity.
"""
from __future__ import annotations

import math

import numpy as np
import pytest

import oracle
from oracle import merge as M
from paper_2102_08862_b200 import gen

import merge_eval as ME

CB = 1.0 / 666.7


def _local(X, Y, Phi, alpha):
    """Global point / direction -> local frame of a sector whose axis points at angle alpha (generator convention)."""
    return (X * math.cos(alpha) + Y * math.sin(alpha), -X * math.sin(alpha) + Y * math.cos(alpha), math.sin(Phi - alpha))


@pytest.mark.parametrize("side_sign", [1, -1])
@pytest.mark.parametrize("Phi_deg,k", [(35.0, 1.7), (52.0, -0.8), (41.0, 0.0), (28.0, 3.1)])
def test_MR_rotation_matches_the_global_frame(side_sign, Phi_deg, k):
    p = M.default_merge_params()
    alpha = math.radians(30.0)                       # sector 1; neighbours at 50 and 10 degrees
    alpha2 = alpha + side_sign * math.radians(20.0)
    Phi = math.radians(Phi_deg)
    # a point near the sector edge on that side, 150 cm from the beam axis
    ang = alpha + side_sign * math.radians(9.0)
    X, Y = 150.0 * math.cos(ang), 150.0 * math.sin(ang)
    x, y, s = _local(X, Y, Phi, alpha)
    st = M.rotate(p, [x, y, 12.5, s, 0.3, k], side_sign)
    x2, y2, s2 = _local(X, Y, Phi, alpha2)
    assert abs(st[0] - x2) < 2e-4 and abs(st[1] - y2) < 2e-4 and abs(st[3] - s2) < 2e-6
    assert st[2] == np.float32(12.5) and st[4] == np.float32(0.3) and st[5] == np.float32(k)      # z, t, k unchanged
    # there and back
    back = M.rotate(p, st, -side_sign)
    assert abs(back[0] - x) < 2e-4 and abs(back[1] - y) < 2e-4 and abs(back[3] - s) < 2e-6
    # the rotated state, transported, stays on the SAME circle: compare with the exact circle in the new frame (double)
    xn = x2 + 9.0
    ok, tr = M.transport_state(p, st, xn)
    assert ok
    kc = CB * k
    sn = s2 + kc * (xn - x2)
    if k == 0.0:
        y_exact = y2 + (xn - x2) * s2 / math.sqrt(1 - s2 * s2)
        arc = (xn - x2) / math.sqrt(1 - s2 * s2)
    else:
        y_exact = y2 + (math.sqrt(1 - s2 * s2) - math.sqrt(1 - sn * sn)) / kc
        arc = (math.asin(sn) - math.asin(s2)) / kc
    assert abs(tr[1] - y_exact) < 3e-4 and abs(tr[3] - sn) < 2e-6 and abs(tr[2] - (12.5 + 0.3 * arc)) < 3e-4


def test_MR_sector_angle_constants_are_twenty_degrees():
    """Cd, Sd come from tan(10 deg) without libm: rotating (1, 0) must give (cos 20, -sin 20)."""
    p = M.default_merge_params()
    st = M.rotate(p, [1.0, 0.0, 0.0, 0.0, 0.0, 0.0], 1)
    assert abs(st[0] - math.cos(math.radians(20.0))) < 1e-7 and abs(st[1] + math.sin(math.radians(20.0))) < 1e-7
    assert abs(st[3] + math.sin(math.radians(20.0))) < 1e-7


def test_MT_state_transport_is_the_state_part_of_the_C5_transport():
    rng = np.random.default_rng(5)
    p = M.default_merge_params()
    tp = oracle.default_params()
    n_ok = 0
    for _ in range(400):
        s0 = rng.uniform(-0.9, 0.9)
        st = [rng.uniform(85, 240), rng.uniform(-30, 30), rng.uniform(-50, 50), s0, rng.uniform(-1.2, 1.2), rng.uniform(-6, 6)]
        xn = st[0] + rng.uniform(-60, 60)
        ok_m, a = M.transport_state(p, st, xn)
        ok_f, b, _ = oracle.transport(tp, st, [1, 0, 0.1, 0, 0, 100, 1, 0, 0.1], xn)
        assert ok_m == ok_f
        np.testing.assert_array_equal(a, b)
        n_ok += ok_m
    assert n_ok > 200


_cache = {}


def _tracked(cid, seed, **kw):
    key = (cid, seed, tuple(sorted(kw.items())))
    if key not in _cache:
        c = gen.preset(cid, seed)
        for k, v in kw.items():
            setattr(c, k, v)
        tf = gen.generate(c)
        res = oracle.track(oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(max(c.sigma_y_cm, 0.08), max(c.sigma_z_cm, 0.12)),
                           tf.row, tf.pad, tf.time)
        mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
        _cache[key] = (tf, res, mr)
    return _cache[key]


def _evaluate(tf, res, mr):
    keys = ME.track_truth_keys(tf, res.tr_hit_offset, res.tr_n_hits, res.tr_hit_index)
    return ME.evaluate_links(keys, res.tr_sector, res.tr_first_row, res.tr_last_row, mr.next)


def test_MH_noise_free_helices_crossing_boundaries_are_linked_and_nothing_else():
    tf, res, mr = _tracked(1, 4, fixed_tracks=600, sigma_y_cm=0.0, sigma_z_cm=0.0, dropout=0.0, noise_frac=0.0, pt_min=0.15)
    rep = _evaluate(tf, res, mr)
    assert rep["expected"] >= 150, rep
    assert rep["got"] == rep["expected"], rep
    assert rep["wrong"] == 0, rep
    # chains: a particle crossing two boundaries gives a chain of three pieces with one root
    assert (np.bincount(mr.root, minlength=len(mr.root)) >= 3).any()


@pytest.mark.parametrize("seed", [1, 2])
def test_MI_invariants(seed):
    tf, res, mr = _tracked(1, seed)
    n = len(res.tr_seed)
    a = np.where(mr.next >= 0)[0]
    b = mr.next[a]
    assert mr.n_links == a.size and mr.n_links > 1000
    np.testing.assert_array_equal(mr.prev[b], a)                                   # reciprocal
    assert np.unique(b).size == b.size                                             # a track continues at most one track
    sa, sb = res.tr_sector[a], res.tr_sector[b]
    assert np.all(sa // 18 == sb // 18) and np.all(np.isin((sa % 18 - sb % 18) % 18, (1, 17)))   # adjacent, same side
    rb = np.rint((res.tr_par[b, 0].astype(np.float64) - 85.0) / 1.07).astype(np.int64)     # row the state of B sits on
    assert np.all(rb <= res.tr_first_row[b]) and np.all(rb > res.tr_first_row[a])
    assert np.all(rb >= res.tr_last_row[a] - 1) and np.all(rb <= res.tr_last_row[a] + 13)
    # roots: fixed points of prev, and every chain member points at its chain's first piece
    assert np.all(mr.prev[mr.root] == -1)
    np.testing.assert_array_equal(mr.root[b], mr.root[a])
    np.testing.assert_array_equal(mr.root[np.where(mr.prev < 0)[0]], np.where(mr.prev < 0)[0])
    assert n - mr.n_links == np.unique(mr.root).size                               # merged tracks = tracks - links


def test_MP_result_does_not_depend_on_the_input_order():
    tf, res, mr = _tracked(1, 1)
    n = len(res.tr_seed)
    perm = np.random.default_rng(11).permutation(n)
    m2 = M.merge(M.default_merge_params(36), res.tr_seed[perm], res.tr_sector[perm], res.tr_first_row[perm],
                 res.tr_last_row[perm], res.tr_par[perm])
    seed_next = np.where(mr.next >= 0, res.tr_seed[np.maximum(mr.next, 0)], -1)
    seed_next2 = np.where(m2.next >= 0, res.tr_seed[perm][np.maximum(m2.next, 0)], -1)
    np.testing.assert_array_equal(seed_next[perm], seed_next2)


@pytest.mark.parametrize("seed", [1, 2])
def test_ME_link_efficiency_and_purity_on_config1(seed):
    tf, res, mr = _tracked(1, seed)
    rep = _evaluate(tf, res, mr)
    assert rep["expected"] >= 2000, rep
    assert rep["efficiency"] >= 0.97, rep
    assert rep["wrong_rate"] <= 0.02, rep


@pytest.mark.parametrize("seed", [1, 2])
def test_MV_vertex_time_and_offset_against_generator_truth(seed):
    """C9: a primary track transported to the beam line arrives at time (t0 v + L - side z_v) / Z with |y| ~ 0."""
    tf, res, mr = _tracked(1, seed)
    ok, vt, vy = M.vertex_time(M.default_merge_params(36), res.tr_par)
    keys = ME.track_truth_keys(tf, res.tr_hit_offset, res.tr_n_hits, res.tr_hit_index)
    tr = tf.tracks[np.where(keys >= 0, keys // (64 * 16), 0)]
    side = np.where(res.tr_sector < 18, 1.0, -1.0)
    t_true = (tr["t0_us"] * 2.58 + 250.0 - side * tr["z_v"]) / 0.516
    sel = (keys >= 0) & (keys % 16 == 0) & (mr.prev < 0) & (tr["pt"] > 0.3)          # first outgoing arc, innermost piece
    assert sel.sum() > 2000 and np.all(ok[sel] == 1)
    d = (vt - t_true)[sel]
    assert abs(np.median(d)) < 0.02 and np.median(np.abs(d)) < 0.15 and np.percentile(np.abs(d), 99) < 1.0, (np.median(d), np.median(np.abs(d)))
    assert np.median(np.abs(vy[sel])) < 0.2 and np.percentile(np.abs(vy[sel]), 95) < 1.0
    # a state that cannot reach x = 0 below sin_phi_max is flagged and zeroed
    st = np.array([[150.0, 0.0, 0.0, 0.5, 0.2, 8.0, 100.0]], np.float32)                # s - k cB x = 0.5 - 1.8 < -0.95
    ok1, t1, y1 = M.vertex_time(M.default_merge_params(36), st)
    assert ok1[0] == 0 and t1[0] == 0.0 and y1[0] == 0.0


def test_degenerate_inputs():
    p = M.default_merge_params(36)
    e = M.merge(p, [], [], [], [], np.zeros((0, 7), np.float32))
    assert e.n_links == 0 and e.next.size == 0
    # a single-sector geometry has no neighbours
    tf, res, mr = _tracked(1, 1)
    one = M.merge(M.default_merge_params(1), res.tr_seed, np.zeros_like(res.tr_sector), res.tr_first_row, res.tr_last_row, res.tr_par)
    assert one.n_links == 0 and np.all(one.next == -1) and np.array_equal(one.root, np.arange(len(res.tr_seed)))


def _pair_across_boundary(state_row_b, first_row_b, state_row_a=40, first_row_a=40, last_row_a=99):
    """Two hand-made tracks on ONE straight radial line through the boundary between sectors 0 and 1: A in sector 0
    (rows first_row_a..last_row_a), B in sector 1; each state is the exact line at the row it claims to sit on."""
    x0, pitch = 85.0, 1.07
    T = math.tan(math.radians(10.0))
    Phi = math.radians(17.0)                                  # global direction; the line passes the boundary (20 deg) near row 100
    xa = x0 + pitch * state_row_a
    # global line through the point P = 192 cm * (cos 20, sin 20) with direction Phi
    P = (192.0 * math.cos(math.radians(20.0)), 192.0 * math.sin(math.radians(20.0)))
    def local_state(alpha_deg, x_local):
        al = math.radians(alpha_deg)
        px, py, ph = _local(P[0], P[1], Phi, al)
        tanl = math.tan(Phi - al)
        return [x_local, py + (x_local - px) * tanl, 0.0, math.sin(Phi - al), 0.0, 0.0, 100.0]
    a = local_state(10.0, xa)
    b = local_state(30.0, x0 + pitch * state_row_b)
    par = np.array([a, b], np.float32)
    return ([11, 22], [0, 1], [first_row_a, first_row_b], [last_row_a, 140], par)


def test_MC_a_state_above_its_first_row_is_never_a_continuation_and_chains_are_acyclic():
    """Reading M7: B is a candidate only if its state sits at its inner end (r_B <= f_B) and above A's own state row."""
    p = M.default_merge_params(36)
    ok = M.merge(p, *_pair_across_boundary(state_row_b=101, first_row_b=101))
    assert ok.n_links == 1 and ok.next[0] == 1 and ok.prev[1] == 0 and ok.root[1] == 0
    # the same B, but its hits start at row 95 and its state (failed down refit) stayed on row 101: not a candidate
    bad = M.merge(p, *_pair_across_boundary(state_row_b=101, first_row_b=95))
    assert bad.n_links == 0 and np.all(bad.next == -1) and np.array_equal(bad.root, [0, 1])
    # A's own state sits ABOVE the candidate's row (A's refit failed part-way, state on row 105): r_B > r_A fails
    bad2 = M.merge(p, *_pair_across_boundary(state_row_b=101, first_row_b=101, state_row_a=105))
    assert bad2.n_links == 0
    # real data: along every chain the state rows strictly increase
    tf, res, mr = _tracked(1, 1)
    rs = np.floor((res.tr_par[:, 0] - np.float32(85.0)) / np.float32(1.07) + np.float32(0.5)).astype(np.int64)
    a = np.where(mr.next >= 0)[0]
    assert np.all(rs[mr.next[a]] > rs[a]) and np.all(rs[mr.next[a]] <= res.tr_first_row[mr.next[a]])
    assert (rs > res.tr_first_row).sum() >= 1            # the input does hold tracks whose state is not at the inner end


# ----------------------------------------------------------------------------- C10: central-electrode merging
def _ce_pair(x_c=150.0, t_a=0.4, rows_a=(40, 58), row_b=63, sec_a=3, slope=0.05, k=0.0, t_b=None, shift_b=0.0):
    """Two hand-made tracks on ONE straight line of the common local frame of sectors sec_a / sec_a + 18: A holds rows
    rows_a with its state on its first row, B starts on row_b in the mirror sector.  The time-derived coordinate rises with
    slope t_a per unit path up to the crossing at x = x_c and falls with the mirrored slope behind it."""
    x0, pitch = 85.0, 1.07
    ds_dx = math.sqrt(1.0 + slope * slope)            # path per unit x of a straight line
    s = slope / ds_dx
    xa, xb = x0 + pitch * rows_a[0], x0 + pitch * row_b
    z_of = lambda x: (x - x_c) * ds_dx * t_a if x <= x_c else -(x - x_c) * ds_dx * t_a     # relative to the crossing, cm
    t_cross = 5000.0                                  # time coordinate of the crossing [bins]
    tb = -t_a if t_b is None else t_b
    a = [xa, slope * xa, 0.0, s, t_a, k, t_cross + z_of(xa) / 0.516]                       # z_rel = 0 at its own time_ref
    b = [xb, slope * xb, 0.0, s, tb, k, t_cross + (z_of(xb) + shift_b) / 0.516]
    par = np.array([a, b], np.float32)
    return ([11, 22], [sec_a, (sec_a + 18) % 36], [rows_a[0], row_b], [rows_a[1], 140], par), t_cross


def test_CEL_mirrored_line_is_linked_and_the_crossing_time_is_the_closed_form():
    p = M.default_ce_params(36)
    for x_c in (149.0, 150.5, 152.0):                 # anywhere between A's last row (x = 147.06) and B's state (x = 152.41)
        args, t_cross = _ce_pair(x_c=x_c)
        r = M.merge_ce(p, *args)
        assert r.n_links == 1 and r.next[0] == 1 and r.prev[1] == 0 and r.next[1] == -1
        assert abs(float(r.t_ce[0]) - t_cross) < 2e-3 and r.t_ce[1] == 0.0
    # a C-side track that crosses to the A side links the same way (the mirror of sector 21 is sector 3)
    args, t_cross = _ce_pair(sec_a=21)
    r = M.merge_ce(p, *args)
    assert r.n_links == 1 and abs(float(r.t_ce[0]) - t_cross) < 2e-3


def test_CES_sign_mirror_and_interval_conditions():
    p = M.default_ce_params(36)
    link = lambda **kw: M.merge_ce(p, *_ce_pair(**kw)[0]).n_links
    assert link() == 1
    assert link(t_a=-0.4) == 0                        # CE2: a track moving away from the electrode cannot cross it
    assert link(t_b=0.4) == 0                         # the slope behind the electrode must be mirrored (dt = t_A + t_B)
    assert link(t_b=-0.35) == 1 and link(t_b=-0.25) == 0          # ... within cut_dzds = 0.1
    assert link(x_c=140.0) == 0                       # crossing 7 cm BEFORE A's last row: dzm exceeds twice the gap advance by > 2 cm
    # the allowed interval of dzm is [0, 2 * 0.4 * 5.36] = [0, 4.28] cm and dzm = 1.93 cm here; |ez| < cut_z = 2 cm beyond it
    assert link(shift_b=3.5) == 1 and link(shift_b=4.5) == 0 and link(shift_b=-4.0) == 1 and link(shift_b=-5.0) == 0
    # same sector pairing only: B in a different phi slice does not link
    args, _ = _ce_pair()
    args[1][1] = 22
    assert M.merge_ce(p, *args).n_links == 0
    assert M.merge_ce(M.default_ce_params(18), *_ce_pair()[0]).n_links == 0       # half a TPC has no mirror sectors


def _ce_expected(res, keys):
    """Pairs (i, j) of tracks that belong to the same (particle, arc), sit in mirror sectors and satisfy C10's row window."""
    from collections import defaultdict
    groups = defaultdict(list)
    for i, k in enumerate(keys):
        if k >= 0:
            groups[(k // (64 * 16), k % 16)].append(i)
    exp = set()
    for v in groups.values():
        for i in v:
            for j in v:
                if (res.tr_sector[j] == (res.tr_sector[i] + 18) % 36 and res.tr_par[i, 4] > 0 and
                        res.tr_last_row[i] - 1 <= res.tr_first_row[j] <= res.tr_last_row[i] + 13 and res.tr_first_row[j] > res.tr_first_row[i]):
                    exp.add((i, j))
    return exp


def _ce_frame(seed, noise_free):
    c = gen.preset(1, seed)
    c.fixed_tracks, c.zv_sigma_cm, c.eta_max, c.pt_min = 3000, 30.0, 0.3, 0.3      # many tracks through the electrode INSIDE the TPC
    if noise_free:
        c.sigma_y_cm = c.sigma_z_cm = c.dropout = c.noise_frac = 0.0
    tf = gen.generate(c)
    res = oracle.track(oracle.default_geometry(36, tf.max_time_bin), oracle.default_params(), tf.row, tf.pad, tf.time)
    return tf, res, M.merge_ce(M.default_ce_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)


def test_CEH_noise_free_helices_through_the_electrode_and_CET_crossing_time():
    tf, res, r = _ce_frame(3, noise_free=True)
    keys = ME.track_truth_keys(tf, res.tr_hit_offset, res.tr_n_hits, res.tr_hit_index)
    a = np.where(r.next >= 0)[0]
    got = set(zip(a.tolist(), r.next[a].tolist()))
    exp = _ce_expected(res, keys)
    assert len(exp) >= 250
    assert got <= exp, "a link that generator truth does not have"
    assert len(got) >= 0.95 * len(exp), (len(got), len(exp))
    # CE-T: the crossing time is the collision time: (t0 v_drift + drift length) / time bin
    tr = tf.tracks[keys[a] // (64 * 16)]
    t_true = (tr["t0_us"] * 2.58 + 250.0) / 0.516
    err = np.abs(r.t_ce[a] - t_true)
    assert np.median(err) < 1e-4 and np.mean(err < 0.05) > 0.98 and err.max() < 1.5       # a crossing inside the last rows of A is clamped to the interval
    assert np.all(r.t_ce[r.next < 0] == 0.0)


def test_CEI_invariants_CEP_order_independence_and_purity_with_noise():
    tf, res, r = _ce_frame(4, noise_free=False)
    keys = ME.track_truth_keys(tf, res.tr_hit_offset, res.tr_n_hits, res.tr_hit_index)
    a = np.where(r.next >= 0)[0]
    b = r.next[a]
    assert r.n_links == a.size >= 150
    np.testing.assert_array_equal(r.prev[b], a)
    assert np.unique(b).size == b.size
    np.testing.assert_array_equal(res.tr_sector[b], (res.tr_sector[a] + 18) % 36)
    assert np.all(res.tr_par[a, 4] > 0)
    rs = np.floor((res.tr_par[:, 0] - np.float32(85.0)) / np.float32(1.07) + np.float32(0.5)).astype(np.int64)
    assert np.all(rs[b] > rs[a]) and np.all(rs[b] <= res.tr_first_row[b]) and np.all(rs[b] >= res.tr_last_row[a] - 1)
    exp = _ce_expected(res, keys)
    got = set(zip(a.tolist(), b.tolist()))
    assert len(got & exp) >= 0.85 * len(exp), (len(got & exp), len(exp))
    assert len(got - exp) <= 0.03 * len(got), (len(got - exp), len(got))
    tr = tf.tracks[np.maximum(keys[a], 0) // (64 * 16)]
    ok = np.array([(i, j) in exp for i, j in zip(a, b)])
    t_true = (tr["t0_us"] * 2.58 + 250.0) / 0.516
    assert np.median(np.abs(r.t_ce[a] - t_true)[ok]) < 0.5
    # order independence
    perm = np.random.default_rng(5).permutation(len(res.tr_seed))
    r2 = M.merge_ce(M.default_ce_params(36), res.tr_seed[perm], res.tr_sector[perm], res.tr_first_row[perm], res.tr_last_row[perm], res.tr_par[perm])
    s1 = np.where(r.next >= 0, res.tr_seed[np.maximum(r.next, 0)], -1)
    s2 = np.where(r2.next >= 0, res.tr_seed[perm][np.maximum(r2.next, 0)], -1)
    np.testing.assert_array_equal(s1[perm], s2)
    np.testing.assert_array_equal(r.t_ce[perm], r2.t_ce)


def test_MD_every_term_of_the_match_distance_decides():
    """d2 = dy^2 wy + dz^2 wz + ds^2 ws + dk^2 wk: two candidates B1, B2 that differ from the extrapolated A in ONE quantity
    only (B2 closer); whichever term it is, A must pick B2 -- and B1 when the roles are swapped."""
    p = M.default_merge_params(36)
    base = _pair_across_boundary(state_row_b=101, first_row_b=101)
    par_a, par_b = base[4][0], base[4][1]
    for col, d1, d2 in ((1, 0.9, 0.3), (2, 0.9, 0.3), (3, 0.03, 0.01), (5, 0.3, 0.1)):        # y, z, sin phi, q/pT
        for swap in (False, True):
            b1, b2 = par_b.copy(), par_b.copy()
            b1[col] += d1
            b2[col] += d2
            if swap:
                b1, b2 = b2, b1
            par = np.array([par_a, b1, b2], np.float32)
            r = M.merge(p, [11, 22, 33], [0, 1, 1], [40, 101, 101], [99, 140, 140], par)
            assert r.next[0] == (1 if swap else 2), (col, swap, r.next)
            assert r.n_links == 1 and r.prev[r.next[0]] == 0


# ---- pins from the line-by-line mutation sweep of the merge oracle -------------------------------------------

def test_MW_the_weights_are_one_over_the_squared_cuts():
    """Two candidates that miss in DIFFERENT quantities: which one wins is decided by w = 1 / cut^2 (cuts chosen so that
    cut^2 differs from 2 cut for every one of them)."""
    p = M.default_merge_params(36)
    p.cut_y_cm, p.cut_z_cm, p.cut_sin_phi, p.cut_q_pt = 1.0, 3.0, 0.05, 0.5
    base = _pair_across_boundary(state_row_b=101, first_row_b=101)
    par_a, par_b = base[4][0], base[4][1]
    # (column, offset) of candidate 1 and of candidate 2; in units of its cut:  0.60 vs 0.50, so candidate 2 wins every time
    y, z, s, k = (1, 1.0), (2, 3.0), (3, 0.05), (5, 0.5)
    for (c1, cut1), (c2, cut2) in ((y, z), (z, y), (y, s), (s, y), (z, k), (k, z), (s, k), (k, s)):
        b1, b2 = par_b.copy(), par_b.copy()
        b1[c1] += 0.60 * cut1
        b2[c2] += 0.50 * cut2
        r = M.merge(p, [11, 22, 33], [0, 1, 1], [40, 101, 101], [99, 140, 140], np.array([par_a, b1, b2], np.float32))
        assert r.next[0] == 2 and r.n_links == 1, (c1, c2, r.next)
        r = M.merge(p, [11, 33, 22], [0, 1, 1], [40, 101, 101], [99, 140, 140], np.array([par_a, b2, b1], np.float32))
        assert r.next[0] == 1, (c1, c2, r.next)


def test_M0_track_index_zero_is_a_track_like_any_other():
    """Index 0 as the better of two candidates, as the link target, and as the better of two predecessors (C7 and C10)."""
    p = M.default_merge_params(36)
    base = _pair_across_boundary(state_row_b=101, first_row_b=101)
    par_a, par_b = base[4][0], base[4][1]
    worse = par_b.copy(); worse[1] += 0.9
    # B (good) at index 0, a worse B' at 1, A at 2: A -> 0
    r = M.merge(p, [22, 33, 11], [1, 1, 0], [101, 101, 40], [140, 140, 99], np.array([par_b, worse, par_a], np.float32))
    assert r.next[2] == 0 and r.prev[0] == 2 and r.n_links == 1 and r.root[0] == 2
    # two predecessors compete for one B: the better A at index 0, a worse A' (shifted in y) at 1
    a_worse = par_a.copy(); a_worse[1] += 0.9
    r = M.merge(p, [11, 12, 22], [0, 0, 1], [40, 40, 101], [99, 99, 140], np.array([par_a, a_worse, par_b], np.float32))
    assert r.next[0] == 2 and r.prev[2] == 0 and r.next[1] == -1
    # C10: the continuation at index 0
    pc = M.default_ce_params(36)
    args, t_cross = _ce_pair()
    seed, sec, fr, lr, par = args
    r = M.merge_ce(pc, seed[::-1], sec[::-1], fr[::-1], lr[::-1], par[::-1].copy())
    assert r.n_links == 1 and r.next[1] == 0 and r.prev[0] == 1 and abs(float(r.t_ce[1]) - t_cross) < 2e-3
    # C10: the better of two continuations at index 0 (the worse one 1 cm off in y)
    b_worse = par[1].copy(); b_worse[1] += 1.0
    r = M.merge_ce(pc, [22, 33, 11], [sec[1], sec[1], sec[0]], [fr[1], fr[1], fr[0]], [lr[1], lr[1], lr[0]], np.array([par[1], b_worse, par[0]], np.float32))
    assert r.next[2] == 0 and r.n_links == 1


def test_CEW_every_term_of_the_electrode_match_distance_adds():
    """C10's d2 = dy^2 wy + ez^2 wz + ds^2 ws + dk^2 wk + dt^2 wt with w = 1 / cut^2: candidates that miss in different
    quantities, 0.6 against 0.5 of the cut."""
    pc = M.default_ce_params(36)
    args, _ = _ce_pair()
    seed, sec, fr, lr, par = args
    cuts = {1: float(pc.cut_y_cm), 3: float(pc.cut_sin_phi), 5: float(pc.cut_q_pt), 4: float(pc.cut_dzds)}
    cols = list(cuts)
    for c1 in cols:
        for c2 in cols:
            if c1 == c2:
                continue
            b1, b2 = par[1].copy(), par[1].copy()
            b1[c1] += 0.60 * cuts[c1]
            b2[c2] += 0.50 * cuts[c2]
            r = M.merge_ce(pc, [11, 22, 33], [sec[0], sec[1], sec[1]], [fr[0], fr[1], fr[1]], [lr[0], lr[1], lr[1]], np.array([par[0], b1, b2], np.float32))
            assert r.next[0] == 2 and r.n_links == 1, (c1, c2, r.next)
    # the time term: B shifted along z until dzm (1.93 cm unshifted, allowed interval [0, 4.28]) is -1.2 cm: ez = -1.2 = 0.6 cut_z;
    # a candidate 0.5 cut_y off wins against it, one 0.7 cut_y off loses
    (s1, s_, f_, l_, par1), _ = _ce_pair(shift_b=1.93 + 0.6 * float(pc.cut_z_cm))
    for off, winner in ((0.5, 2), (0.7, 1)):
        b2 = par[1].copy(); b2[1] += off * float(pc.cut_y_cm)
        r = M.merge_ce(pc, [11, 22, 33], [sec[0], sec[1], sec[1]], [fr[0], fr[1], fr[1]], [lr[0], lr[1], lr[1]], np.array([par[0], par1[1], b2], np.float32))
        assert r.next[0] == winner, (off, r.next)


def test_CERW_row_window_of_the_electrode_merger():
    """l_A + 1 - overlap <= r_B <= l_A + 1 + gap with r_B = floor((x_B - x0) / pitch + 0.5): the edges, with A ending on row 58."""
    pc = M.default_ce_params(36)
    gap, over = int(pc.max_row_gap), int(pc.max_row_overlap)
    link = lambda row_b: M.merge_ce(pc, *_ce_pair(row_b=row_b, x_c=85.0 + 1.07 * 58.5)[0]).n_links
    assert link(58 + 1 + gap) == 1 and link(58 + 2 + gap) == 0
    assert link(58 + 1 - over) == 1 and link(58 - over) == 0
    # half a TPC (18 sectors) has no mirror sectors but does merge across sector boundaries
    p18 = M.default_merge_params(18)
    base = _pair_across_boundary(state_row_b=101, first_row_b=101)
    assert M.merge(p18, *base).n_links == 1


def test_M7A_the_continuation_must_lie_above_the_state_row_of_A_and_index_zero_as_a_predecessor_in_C10():
    """M7: r_B > max(f_A, r_A) with r_A the row A's state sits on -- which is above f_A when the down refit failed early."""
    p = M.default_merge_params(36)
    link = lambda rb: M.merge(p, *_pair_across_boundary(state_row_b=rb, first_row_b=rb, state_row_a=60, first_row_a=40, last_row_a=61)).n_links
    assert link(60) == 0 and link(61) == 1              # row 60 is inside the row window [60, 74] but not above A's state row
    pc = M.default_ce_params(36)
    for state_row, linked in ((58, 1), (59, 0)):        # C10 likewise: A (rows 40 .. 58) with its state on row 58 / on r_B = 59
        (seed, sec, fr, lr, par), _ = _ce_pair(rows_a=(state_row, 58), row_b=59)
        assert M.merge_ce(pc, seed, sec, [40, fr[1]], lr, par).n_links == linked, state_row
    # two tracks compete to continue into one B behind the electrode: the better one has index 0
    (seed, sec, fr, lr, par), _ = _ce_pair()
    a_worse = par[0].copy(); a_worse[1] += 1.0
    r = M.merge_ce(pc, [11, 12, 22], [sec[0], sec[0], sec[1]], [fr[0], fr[0], fr[1]], [lr[0], lr[0], lr[1]], np.array([par[0], a_worse, par[1]], np.float32))
    assert r.next[0] == 2 and r.prev[2] == 0 and r.next[1] == -1 and r.n_links == 1
