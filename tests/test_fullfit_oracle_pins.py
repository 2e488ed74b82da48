"""Pins of the C12 oracle (oracle/tpc_oracle.cpp::orc_refit_full: Kalman refit with the full 5x5 covariance, multiple
scattering and energy loss).

The paper prints nothing for this step, so the pins are what the mathematics fixes:
  FF-J  every entry of the transport Jacobian against the numerical derivative of the exact helix (fp64, asin / cos forms),
  FF-Q  the process noise of a scattering step against a Monte-Carlo of random 3-D kinks, and theta0 against the textbook
        13.6 MeV / (beta p) * sqrt(x / X0),
  FF-E  the accumulated energy-loss correction against the integrated dp/dl = dE/dx / beta,
  FF-G  on a straight line the filter with process noise is the Bayesian linear regression with correlated noise (brute force),
  FF-0  without material and without dip it reproduces the block fit of C5 / C8 (pinned by K1..K3),
  FF-P  on tracks simulated WITH scattering and energy loss the pull of q/pT is unit-width with the material and too wide without,
  FF-N / FF-I  generator data: consistent with C8, bookkeeping.
"""
from __future__ import annotations

import math
from types import SimpleNamespace

import numpy as np
import pytest

import oracle
from oracle import merge as M
from paper_2102_08862_b200 import gen

NO_MATERIAL = (0.0, 0.0, 0.13957, 0.0)
Y, Z, S, T, K = range(5)


def tri(i, j):
    return i * (i + 1) // 2 + j if i >= j else j * (j + 1) // 2 + i


def full(cov15):
    return np.array([[cov15[tri(i, j)] for j in range(5)] for i in range(5)], np.float64)


def pack(Pm):
    return [Pm[i][j] for i in range(5) for j in range(i + 1)]


def helix_exact(v, dx, cB):
    """(y, z, s, t, k) at x -> the same at x + dx on the exact helix, fp64."""
    y, z, s, t, k = v
    kap = cB * k
    sn = s + kap * dx
    c, cn = math.sqrt(1 - s * s), math.sqrt(1 - sn * sn)
    if abs(kap) < 1e-12:
        return np.array([y + dx * s / c, z + t * dx / c, sn, t, k])
    return np.array([y + (c - cn) / kap, z + t * (math.asin(sn) - math.asin(s)) / kap, sn, t, k])


@pytest.mark.parametrize("state,dx", [
    ((3.0, 10.0, 0.30, 0.60, 2.0), -1.07), ((-5.0, 40.0, -0.55, -0.90, -4.0), -1.07), ((1.0, 0.0, 0.10, 1.20, 6.0), -3.21),
    ((7.0, 5.0, 0.70, 0.30, -1.0), 1.07), ((0.0, 0.0, -0.20, -1.50, 0.5), -10.7)])
def test_FFJ_transport_jacobian_is_the_derivative_of_the_exact_helix(state, dx):
    p = oracle.default_params()
    cB = float(p.inv_R_per_qpt)
    x0 = 150.0
    F = np.zeros((5, 5))
    for j in range(5):                                 # P = e_j e_j^T  ->  P' = F[:, j] F[:, j]^T, and F[j][j] = 1
        P0 = np.zeros((5, 5)); P0[j, j] = 1.0
        ok, st, cv = oracle.full_step(p, [x0, *state], pack(P0), x0 + dx, NO_MATERIAL)
        assert ok
        F[:, j] = full(cv)[:, j]
    Fn = np.zeros((5, 5))
    v0 = np.array(state, np.float64)
    for j in range(5):
        h = 1e-6 * max(1.0, abs(v0[j]))
        a, b = v0.copy(), v0.copy()
        a[j] += h; b[j] -= h
        Fn[:, j] = (helix_exact(a, dx, cB) - helix_exact(b, dx, cB)) / (2 * h)
    # state itself
    np.testing.assert_allclose(st[1:], helix_exact(v0, dx, cB), rtol=2e-6, atol=2e-5)
    exact = [(Y, Y), (Z, Z), (S, S), (T, T), (K, K), (Y, S), (Y, K), (S, K), (Z, T)]
    for (a, b) in exact:
        assert abs(F[a, b] - Fn[a, b]) <= 2e-4 * max(abs(Fn[a, b]), 1e-3), (a, b, F[a, b], Fn[a, b])
    for (a, b) in [(Z, S), (Z, K)]:                    # derivative of the chord, not of the arc (reading FF2): off by about (sn - s) / (3 (s + sn))
        assert abs(F[a, b] - Fn[a, b]) <= 8e-2 * abs(Fn[a, b]) + 1e-7, (a, b, F[a, b], Fn[a, b])
        assert F[a, b] * Fn[a, b] > 0
    zero = [(a, b) for a in range(5) for b in range(5) if (a, b) not in exact + [(Z, S), (Z, K)]]
    for (a, b) in zero:
        assert F[a, b] == 0.0 and abs(Fn[a, b]) < 1e-6, (a, b)


def test_FFJ_covariance_propagation_is_F_P_Ft_on_a_dense_matrix():
    p = oracle.default_params()
    rng = np.random.default_rng(5)
    L = rng.normal(size=(5, 5)) * np.array([0.1, 0.2, 0.01, 0.02, 0.3])[:, None]
    P0 = L @ L.T
    state, dx, x0 = (3.0, 10.0, 0.30, 0.60, 2.0), -2.14, 140.0
    F = np.zeros((5, 5))
    for j in range(5):
        E = np.zeros((5, 5)); E[j, j] = 1.0
        F[:, j] = full(oracle.full_step(p, [x0, *state], pack(E), x0 + dx, NO_MATERIAL)[2])[:, j]
    ok, st, cv = oracle.full_step(p, [x0, *state], pack(P0), x0 + dx, NO_MATERIAL)
    np.testing.assert_allclose(full(cv), F @ P0 @ F.T, rtol=2e-5, atol=1e-9)


# ---- FF-Q: process noise of one step -------------------------------------------------------------------------------------

def _noise_of_a_step(state, dx, fp):
    p = oracle.default_params()
    ok, st, cv = oracle.full_step(p, [150.0, *state], [0.0] * 15, 150.0 + dx, fp)
    assert ok
    return st, full(cv)


def test_FFQ_theta0_is_the_textbook_highland_width():
    # p = 1 GeV/c, t = 0 (p = pT), pion: theta0 = 13.6 MeV / (beta p) * sqrt(L / X0); one step of L = 1.07 cm through X0 = 107 cm
    m, pabs = 0.13957, 1.0
    beta = pabs / math.sqrt(pabs * pabs + m * m)
    st, Q = _noise_of_a_step((0.0, 0.0, 0.0, 0.0, 1.0 / pabs), -1.07, (1.0 / 107.0, 0.0, m, 0.0))
    L = 1.07 * (1 + (float(oracle.default_params().inv_R_per_qpt) * 1.07) ** 2 / 24)      # arc of the (nearly straight) step
    theta0 = 0.0136 / (beta * pabs) * math.sqrt(L / 107.0)
    s_new = st[3]
    assert abs(math.sqrt(Q[S, S] / (1 - s_new ** 2)) - theta0) < 2e-4 * theta0            # t = 0: var(s) = theta0^2 cos^2(phi)
    assert abs(math.sqrt(Q[T, T]) - theta0) < 2e-4 * theta0
    assert Q[K, K] == 0.0 and Q[K, T] == 0.0 and Q[Y, Y] == 0.0 and Q[Z, Z] == 0.0        # no dip: a kink leaves q/pT alone
    # scaling: 1 / (beta p)^2 and path length
    st2, Q2 = _noise_of_a_step((0.0, 0.0, 0.0, 0.0, 4.0), -1.07, (1.0 / 107.0, 0.0, m, 0.0))
    p2 = 0.25
    b2 = p2 / math.sqrt(p2 * p2 + m * m)
    assert abs(Q2[T, T] / Q[T, T] - (beta * pabs / (b2 * p2)) ** 2) < 2e-3 * (beta * pabs / (b2 * p2)) ** 2
    st3, Q3 = _noise_of_a_step((0.0, 0.0, 0.0, 0.0, 1.0), -3.21, (1.0 / 107.0, 0.0, m, 0.0))
    assert abs(Q3[T, T] / Q[T, T] - 3.0) < 1e-3


@pytest.mark.parametrize("s0,t0,k0", [(0.3, 0.8, 2.0), (-0.6, -1.4, -5.0), (0.05, 0.2, 0.7)])
def test_FFQ_process_noise_is_the_covariance_of_random_kinks(s0, t0, k0):
    """Monte-Carlo in fp64: kink the 3-D direction by two independent angles of width theta0 in the planes orthogonal to it,
    keep |p|, and look at the scatter of (sin phi, dz/ds, q/pT)."""
    m = 0.13957
    fp = (1.0 / 50.0, 0.0, m, 0.0)
    dx = -2.0 ** -7                                     # a negligible transport (exact in fp32 at x = 150): the noise is evaluated at (s0, t0, k0)
    st, Q = _noise_of_a_step((0.0, 0.0, s0, t0, k0), dx, fp)
    # theta0^2 of that step from the textbook formula
    pt = 1.0 / abs(k0)
    pabs = pt * math.sqrt(1 + t0 * t0)
    beta = pabs / math.sqrt(pabs * pabs + m * m)
    Lp = abs(dx) / math.sqrt(1 - s0 * s0) * math.sqrt(1 + t0 * t0)
    th2 = (0.0136 / (beta * pabs)) ** 2 * Lp / 50.0
    # unit kinks: the covariance scales with theta0^2, so sample with a convenient small width and rescale
    w = 1e-3
    rng = np.random.default_rng(11)
    n = 400000
    a1, a2 = rng.normal(0, w, n), rng.normal(0, w, n)
    phi, lam = math.asin(s0), math.atan(t0)
    d = np.array([math.cos(lam) * math.cos(phi), math.cos(lam) * math.sin(phi), math.sin(lam)])
    e1 = np.array([-math.sin(phi), math.cos(phi), 0.0])
    e2 = np.array([-math.sin(lam) * math.cos(phi), -math.sin(lam) * math.sin(phi), math.cos(lam)])
    dn = d[None, :] + a1[:, None] * e1[None, :] + a2[:, None] * e2[None, :]
    dn /= np.linalg.norm(dn, axis=1)[:, None]
    cl = np.hypot(dn[:, 0], dn[:, 1])
    s1, t1 = dn[:, 1] / cl, dn[:, 2] / cl
    k1 = np.sign(k0) / (pabs * cl)
    C = np.cov(np.stack([s1 - s0, t1 - t0, k1 - k0])) * (th2 / (w * w))
    got = np.array([[Q[a, b] for b in (S, T, K)] for a in (S, T, K)])
    scale = np.sqrt(np.outer(np.diag(C), np.diag(C)))
    assert np.max(np.abs(got - C) / scale) < 0.01, (got, C)
    assert abs(Q[S, T]) == 0.0 and abs(Q[S, K]) == 0.0               # the azimuthal and the dip kink are independent
    assert Q[K, T] * (t0 * k0) > 0                                     # sign of the (t, k) correlation
    assert np.all(Q[[Y, Z], :] == 0.0)


# ---- FF-E: energy loss ----------------------------------------------------------------------------------------------------

@pytest.mark.parametrize("pt,t0", [(0.3, 0.5), (0.15, -1.0), (1.0, 0.1)])
def test_FFE_energy_loss_accumulates_like_the_integrated_stopping_power(pt, t0):
    """Inward over 100 pad rows with a dE/dx a hundred times that of the gas: |p| at the end against dp/dl = (dedx / beta^2) / beta
    integrated in fine steps over the same path length."""
    m, dedx = 0.13957, 1.7e-4
    p = oracle.default_params()
    cB = float(p.inv_R_per_qpt)
    st = np.array([85.0 + 1.07 * 120, 0.0, 0.0, 0.1, t0, 1.0 / pt], np.float32)
    cv = np.zeros(15, np.float32)
    path = 0.0
    pabs = pt * math.sqrt(1 + t0 * t0)
    for r in range(119, 19, -1):
        before = st.astype(np.float64)
        ok, st, cv = oracle.full_step(p, st, cv, 85.0 + 1.07 * r, (0.0, dedx, m, 0.0))
        assert ok
        kap = cB * before[5]
        arc = (math.asin(before[3] + kap * (st[0] - before[0])) - math.asin(before[3])) / kap
        L = abs(arc) * math.sqrt(1 + t0 * t0)
        path += L
        for _ in range(200):                           # the reference integrates with 200 sub-steps per row
            beta = pabs / math.sqrt(pabs * pabs + m * m)
            pabs += (dedx / beta ** 2) / beta * (L / 200)
    p_fit = math.sqrt(1 + t0 * t0) / abs(float(st[5]))
    p_start = pt * math.sqrt(1 + t0 * t0)
    assert p_fit > p_start                              # inward: the momentum comes back
    assert abs((p_fit - p_start) / (pabs - p_start) - 1.0) < 5e-3, (p_fit, pabs, p_start)
    assert (pabs - p_start) / p_start > 0.015           # the effect is large enough to be tested
    assert st[4] == np.float32(t0)                      # dz/ds is untouched
    assert np.all(cv == 0.0)                            # no straggling asked for, no scattering


def test_FFE_straggling_variance_is_the_squared_fraction_of_the_correction():
    m, dedx, frac = 0.13957, 1.7e-4, 0.25
    k0 = 4.0
    st0, Q0 = _noise_of_a_step((0.0, 0.0, 0.1, 0.3, k0), -1.07, (0.0, dedx, m, 0.0))
    st, Q = _noise_of_a_step((0.0, 0.0, 0.1, 0.3, k0), -1.07, (0.0, dedx, m, frac))
    assert st[5] == st0[5] and st[5] < k0
    dk = k0 - float(st[5])
    assert abs(math.sqrt(Q[K, K]) - frac * dk) < 2e-3 * frac * dk
    Q[K, K] = 0.0
    assert np.all(Q == 0.0)


# ---- FF-U / FF-G / FF-0: the update and the filter as a whole --------------------------------------------------------------

def test_FFU_two_scalar_updates_are_the_joint_kalman_update_of_a_dense_covariance():
    rng = np.random.default_rng(3)
    L = rng.normal(size=(5, 5)) * np.array([0.3, 0.4, 0.02, 0.03, 0.5])[:, None]
    P0 = L @ L.T
    v0 = np.array([2.0, -7.0, 0.25, -0.4, 1.5])
    ry, rz = 0.08 ** 2, 0.12 ** 2
    ym, zm = 2.31, -7.42
    st, cv = oracle.full_update([100.0, *v0], pack(P0), ym, zm, ry, rz)
    H = np.zeros((2, 5)); H[0, Y] = 1; H[1, Z] = 1
    Sm = H @ P0 @ H.T + np.diag([ry, rz])
    G = P0 @ H.T @ np.linalg.inv(Sm)
    v1 = v0 + G @ (np.array([ym, zm]) - H @ v0)
    P1 = (np.eye(5) - G @ H) @ P0
    np.testing.assert_allclose(st[1:], v1, rtol=2e-5, atol=2e-6)
    np.testing.assert_allclose(full(cv), P1, rtol=2e-4, atol=1e-8)
    assert st[0] == np.float32(100.0)


def test_FFG_filter_with_scattering_is_the_bayesian_regression_with_correlated_noise():
    """B = 0, no dip, small angles: the model is linear.  Unknowns u = (y_0, s_0, w_0 .. w_{N-2}) with the kink w_l added at row l
    after the transport from row l + 1 (s_l = s_{l+1} + w_l); data = the N hits and the filter's prior at the outermost row."""
    p = oracle.default_params(0.08, 0.12)
    p.inv_R_per_qpt = 0.0
    m = 0.13957
    fp = (1.0 / 100.0, 0.0, m, 0.0)
    rows = [60, 57, 56, 55, 52, 51, 50, 49, 45, 44, 43, 42, 41, 40]         # outermost first, with holes
    x = np.array([85.0 + 1.07 * r for r in rows])
    N = len(x)
    rng = np.random.default_rng(8)
    k0 = 2.5
    y_true = 3.0 + 0.012 * (x - x[-1])
    meas = y_true + rng.normal(0, 0.08, N)
    y_start, s_start = 3.9, 0.02
    st = np.array([x[0], y_start, 0.0, s_start, 0.0, k0], np.float32)
    P0 = np.diag([float(p.c0_y2), float(p.c0_z2), float(p.c0_s2), float(p.c0_t2), float(p.c0_k2)])
    cv = np.array(pack(P0), np.float32)
    q = []
    for i in range(N):
        before = full(cv)[S, S]
        ok, st, cv = oracle.full_step(p, st, cv, float(x[i]), fp)
        assert ok
        q.append(full(cv)[S, S] - before)
        st, cv = oracle.full_update(st, cv, float(meas[i]), 0.0, float(np.float32(0.08) ** 2), float(np.float32(0.12) ** 2))
    # theta0^2 per step from the textbook formula (index i = the step that ENDS on hit i; the first has dx = 0)
    pabs = 1.0 / k0
    beta = pabs / math.sqrt(pabs ** 2 + m ** 2)
    qs = np.array([0.0] + [(0.0136 / (beta * pabs)) ** 2 * abs(x[i] - x[i - 1]) / 100.0 for i in range(1, N)])
    assert np.allclose(q[1:], qs[1:], rtol=0.02)        # (fp32 differences of a variance of 0.1: loose; the regression below is the pin)
    # inner-to-outer numbering for the regression: j = 0 is the innermost hit
    xi, mi, qi = x[::-1], meas[::-1], qs[::-1][:-1]      # qi[l] = kink added on arriving at row l (l = 0 .. N-2)
    nu = 2 + (N - 1)
    rows_A, rhs, var = [], [], []
    for j in range(N):                                  # hit j: y_j = y_0 + (x_j - x_0) s_0 - sum_{l<j} w_l (x_j - x_l)
        a = np.zeros(nu); a[0] = 1; a[1] = xi[j] - xi[0]
        for l in range(j):
            a[2 + l] = -(xi[j] - xi[l])
        rows_A.append(a); rhs.append(mi[j]); var.append(0.08 ** 2)
    a = rows_A[N - 1].copy(); rows_A.append(a); rhs.append(y_start); var.append(float(p.c0_y2))      # prior on y at the outermost row
    a = np.zeros(nu); a[1] = 1; a[2:] = -1.0; rows_A.append(a); rhs.append(s_start); var.append(float(p.c0_s2))   # s_{N-1} = s_0 - sum w
    for l in range(N - 1):                              # priors of the kinks
        a = np.zeros(nu); a[2 + l] = 1; rows_A.append(a); rhs.append(0.0); var.append(max(qi[l], 1e-30))
    A, b, W = np.array(rows_A), np.array(rhs), 1.0 / np.array(var)
    cov_u = np.linalg.inv(A.T @ (W[:, None] * A))
    u = cov_u @ (A.T @ (W * b))
    Pf = full(cv)
    assert abs(st[1] - u[0]) < 3e-4 and abs(st[3] - u[1]) < 3e-5, (st, u[:2])
    assert abs(Pf[Y, Y] / cov_u[0, 0] - 1) < 5e-3 and abs(Pf[S, S] / cov_u[1, 1] - 1) < 5e-3 and abs(Pf[S, Y] / cov_u[1, 0] - 1) < 5e-3
    # and the scattering matters in this set-up: without it the variance of s would be several times smaller
    cov_nomat = np.linalg.inv(A[:N + 2, :2].T @ (W[:N + 2, None] * A[:N + 2, :2]))
    assert cov_u[1, 1] > 2.0 * cov_nomat[1, 1]


def test_FF0_without_material_and_dip_the_fit_is_the_block_filter_of_C5():
    p = oracle.default_params(0.08, 0.12)
    rng = np.random.default_rng(21)
    st_b = np.array([85.0 + 1.07 * 100, 4.0, 1.0, 0.35, 0.0, -3.0], np.float32)
    cv_b = np.array([float(p.c0_y2), 0, float(p.c0_s2), 0, 0, float(p.c0_k2), float(p.c0_z2), 0, float(p.c0_t2)], np.float32)
    st_f = st_b.copy()
    cv_f = np.array(pack(np.diag([float(p.c0_y2), float(p.c0_z2), float(p.c0_s2), float(p.c0_t2), float(p.c0_k2)])), np.float32)
    ry, rz = float(np.float32(0.08) ** 2), float(np.float32(0.12) ** 2)
    for r in range(99, 59, -1):
        xn = 85.0 + 1.07 * r
        okb, st_b, cv_b = oracle.transport(p, st_b, cv_b, xn)
        okf, st_f, cv_f = oracle.full_step(p, st_f, cv_f, xn, NO_MATERIAL)
        assert okb and okf
        ym, zm = float(st_b[1]) + rng.normal(0, 0.08), 1.0 + rng.normal(0, 0.12)
        st_b, cv_b = oracle.update(st_b, cv_b, ym, zm, ry, rz)
        st_f, cv_f = oracle.full_update(st_f, cv_f, ym, zm, ry, rz)
        st_f[4] = 0.0; st_b[4] = 0.0                    # hold the dip at exactly zero: gm = 0, the blocks never couple
    Pf = full(cv_f)
    np.testing.assert_allclose(st_f, st_b, rtol=3e-5, atol=3e-5)
    blk = {(Y, Y): 0, (S, Y): 1, (S, S): 2, (K, Y): 3, (K, S): 4, (K, K): 5, (Z, Z): 6, (T, Z): 7, (T, T): 8}
    for (a, b), i in blk.items():
        assert abs(Pf[a, b] - cv_b[i]) <= 2e-3 * abs(cv_b[i]) + 1e-9, (a, b, Pf[a, b], cv_b[i])
    for a, b in [(Z, Y), (S, Z), (T, Y), (T, S), (K, Z), (K, T)]:
        assert Pf[a, b] == 0.0


@pytest.mark.parametrize("q", [1, -1])
@pytest.mark.parametrize("s0", [-0.6, 0.2, 0.7])
def test_FFR_rotation_scales_row_and_column_s_by_the_derivative_of_the_rotated_sin_phi(q, s0):
    g, p = oracle.default_geometry(), oracle.default_params()
    rng = np.random.default_rng(9)
    L = rng.normal(size=(5, 5)) * np.array([0.2, 0.3, 0.02, 0.03, 0.4])[:, None]
    P0 = (L @ L.T).astype(np.float32).astype(np.float64)
    ok, st, cv = oracle.full_rotate(g, p, [150.0, 20.0, 3.0, s0, 0.4, 1.2], pack(P0), q)
    assert ok
    delta = math.radians(20.0) * q
    f = lambda s: math.sin(math.asin(s) - delta)
    J = (f(s0 + 1e-6) - f(s0 - 1e-6)) / 2e-6
    D = np.diag([1, 1, J, 1, 1])
    np.testing.assert_allclose(full(cv), D @ P0 @ D, rtol=3e-5, atol=1e-10)
    for (a, b) in [(Y, Y), (Z, Y), (Z, Z), (T, Y), (T, Z), (T, T), (K, Y), (K, Z), (K, T), (K, K)]:
        assert full(cv)[a, b] == np.float32(P0[a, b])
    assert abs(st[3] - f(s0)) < 2e-6
    assert abs(st[0] - (150.0 * math.cos(delta) + 20.0 * math.sin(delta))) < 2e-4
    assert abs(st[1] - (-150.0 * math.sin(delta) + 20.0 * math.cos(delta))) < 2e-4
    assert st[2] == 3.0 and st[4] == np.float32(0.4) and st[5] == np.float32(1.2)


# ---- FF-P: tracks simulated WITH scattering and energy loss ---------------------------------------------------------------

def _simulate(n_tracks, fp, seed):
    """Pions of pT 0.12 .. 0.3 GeV/c in sector 0, rows 0 .. 79, stepped row to row on the exact helix in fp64; at every row the
    direction is kinked by theta0 of the segment behind and |p| drops by its energy loss.  Returns clusters, a tracker-like
    result and the true q/pT on row 0."""
    inv_x0, dedx, m, _ = fp
    g = oracle.default_geometry()
    p = oracle.default_params(0.08, 0.12)
    cB = float(p.inv_R_per_qpt)
    rng = np.random.default_rng(seed)
    n_rows_used = 80
    xr = 85.0 + 1.07 * np.arange(152)
    n_pads = np.floor(2.0 * xr * math.tan(math.radians(10.0)) / 0.5)
    row, pad, time, k_true, par, n_hits = [], [], [], [], [], []
    for _ in range(n_tracks):
        pt, q = rng.uniform(0.12, 0.3), rng.choice([-1.0, 1.0])
        s, t, k = rng.uniform(-0.15, 0.15), rng.uniform(-0.8, 0.8), q / pt
        y, zt = rng.uniform(-2, 2), 0.0                 # zt: z relative to the first hit, in cm
        pabs = pt * math.sqrt(1 + t * t)
        k_true.append(k)
        hits = 0
        for r in range(n_rows_used):
            row.append(float(r)); pad.append((y + rng.normal(0, 0.08)) / 0.5 + 0.5 * (n_pads[r] - 1))
            time.append(2000.0 + (zt + rng.normal(0, 0.12)) / 0.516)
            hits += 1
            if r == n_rows_used - 1:
                break
            kap = cB * k
            sn = s + kap * 1.07
            if abs(sn) > 0.9:
                break
            c, cn = math.sqrt(1 - s * s), math.sqrt(1 - sn * sn)
            arc = (math.asin(sn) - math.asin(s)) / kap
            y += (c - cn) / kap; zt += t * arc; s = sn
            Lp = abs(arc) * math.sqrt(1 + t * t)
            beta = pabs / math.sqrt(pabs ** 2 + m ** 2)
            th0 = 0.0136 / (beta * pabs) * math.sqrt(Lp * inv_x0)
            a1, a2 = rng.normal(0, th0), rng.normal(0, th0)
            phi, lam = math.asin(s), math.atan(t)
            phi += a1 / math.cos(lam); lam += a2
            pabs -= (dedx / beta ** 2) / beta * Lp       # outward = with the flight: the momentum drops
            s, t = math.sin(phi), math.tan(lam)
            k = q / (pabs * math.cos(lam))
        n_hits.append(hits)
        # start state of the fit: the true state at the last hit, smeared (the reset covariance is wide)
        par.append([xr[hits - 1], y + rng.normal(0, 0.3), zt + rng.normal(0, 0.3), s + rng.normal(0, 0.02), t + rng.normal(0, 0.02),
                    k * (1 + rng.normal(0, 0.1)), 2000.0])
    n_hits = np.array(n_hits, np.int32)
    off = np.concatenate([[0], np.cumsum(n_hits)[:-1]]).astype(np.int64)
    res = SimpleNamespace(tr_seed=np.arange(n_tracks, dtype=np.int32), tr_sector=np.zeros(n_tracks, np.int32), tr_n_hits=n_hits,
                          tr_hit_offset=off, tr_hit_index=np.arange(int(n_hits.sum()), dtype=np.int32), tr_par=np.array(par, np.float32))
    return g, p, np.array(row, np.float32), np.array(pad, np.float32), np.array(time, np.float32), res, np.array(k_true)


def test_FFP_pull_of_curvature_is_unit_width_with_the_material_and_too_wide_without():
    fp = (1.0 / 300.0, 1.7e-5, 0.13957, 0.0)            # a hundred times the gas' scattering, ten times its stopping power
    g, p, row, pad, time, res, k_true = _simulate(1500, fp, 77)
    none = np.full(len(k_true), -1, np.int32)
    ok, ch, cp, rp, rc = oracle.refit_full(g, p, row, pad, time, res, none, none, fp)
    sel = (ok == 1) & (res.tr_n_hits == 80)
    assert sel.sum() > 1200
    pull = (rp[sel, 5] - k_true[sel]) / np.sqrt(rc[sel, 14])
    width = np.std(pull[np.abs(pull) < 6])
    assert 0.85 < width < 1.2, width
    assert abs(np.mean(pull[np.abs(pull) < 6])) < 0.15
    ok0, _, _, rp0, rc0 = oracle.refit_full(g, p, row, pad, time, res, none, none, NO_MATERIAL)
    pull0 = (rp0[sel, 5] - k_true[sel]) / np.sqrt(rc0[sel, 14])
    assert np.std(pull0[np.abs(pull0) < 30]) > 2.0      # ignoring the material: the quoted error is far too small
    # the energy-loss correction lowers |q/pT| on row 0 by about the momentum the particle lost along the fitted range (about 1 %
    # here), with and without the scattering noise (whose k-dependence leaves a bias of order (sigma_k / k)^2 of its own)
    relk = lambda r: np.median((np.abs(r[sel, 5]) - np.abs(k_true[sel])) / np.abs(k_true[sel]))
    _, _, _, rp_ms, _ = oracle.refit_full(g, p, row, pad, time, res, none, none, (fp[0], 0.0, fp[2], 0.0))
    _, _, _, rp_el, _ = oracle.refit_full(g, p, row, pad, time, res, none, none, (0.0, fp[1], fp[2], 0.0))
    assert 0.003 < relk(rp_ms) - relk(rp) < 0.02, (relk(rp_ms), relk(rp))
    assert 0.003 < relk(rp0) - relk(rp_el) < 0.02, (relk(rp0), relk(rp_el))
    assert abs(relk(rp_el)) < abs(relk(rp0))            # without scattering noise the corrected fit is the less biased one
    # position on row 0 reproduces the innermost hit within its error
    assert np.all(np.abs(rp[sel, 0] - 85.0) < 1e-4)


# ---- FF-N / FF-I: generator data (no material simulated) -----------------------------------------------------------------

_cache = {}


def _frame(cid, seed):
    if (cid, seed) not in _cache:
        c = gen.preset(cid, seed)
        tf = gen.generate(c)
        g = oracle.default_geometry(36, tf.max_time_bin)
        p = oracle.default_params(max(c.sigma_y_cm, 0.08), max(c.sigma_z_cm, 0.12))
        res = oracle.track(g, p, tf.row, tf.pad, tf.time)
        mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
        _cache[(cid, seed)] = (tf, g, p, res, mr)
    return _cache[(cid, seed)]


def test_FFN_on_chains_the_full_fit_agrees_with_the_block_fit_of_C8():
    tf, g, p, res, mr = _frame(1, 1)
    ok8, ch8, cp8, rp8, rc8 = oracle.refit_chains(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev)
    ok, ch, cp, rp, rc = oracle.refit_full(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev, NO_MATERIAL)
    chains = (mr.prev < 0) & (mr.next >= 0)
    both = chains & (ok8 == 1) & (ok == 1)
    assert both.sum() > 2500 and (ok[chains] == 1).mean() > 0.97
    np.testing.assert_array_equal(ch[chains], ch8[chains]); np.testing.assert_array_equal(cp[chains], cp8[chains])
    # the z-(s, k) coupling is the only difference: a small fraction of the error
    dk = np.abs(rp[both, 5] - rp8[both, 5]) / np.sqrt(rc8[both, 5])
    assert np.median(dk) < 0.1 and np.quantile(dk, 0.95) < 0.5, (np.median(dk), np.quantile(dk, 0.95))
    assert np.median(np.abs(rc[both, 14] / rc8[both, 5] - 1)) < 0.05
    assert np.max(np.abs(rp[both, 0] - rp8[both, 0])) < 1e-4
    assert np.quantile(np.abs(rp[both, 1] - rp8[both, 1]), 0.99) < 0.02 and np.quantile(np.abs(rp[both, 2] - rp8[both, 2]), 0.99) < 0.06 and np.median(np.abs(rp[both, 2] - rp8[both, 2])) < 5e-3
    assert np.quantile(np.abs(rp[both, 3] - rp8[both, 3]), 0.99) < 3e-3 and np.quantile(np.abs(rp[both, 4] - rp8[both, 4]), 0.99) < 3e-3
    assert np.median(np.abs(rc[both, 0] / rc8[both, 0] - 1)) < 0.05 and np.median(np.abs(rc[both, 2] / rc8[both, 6] - 1)) < 0.05
    # the gas (default material) changes little at these momenta, but it does change something and never shrinks the errors
    okg, _, _, rpg, rcg = oracle.refit_full(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev)
    bg = both & (okg == 1)
    assert np.mean(rcg[bg, 14] >= rc[bg, 14]) > 0.99 and np.any(rpg[bg, 5] != rp[bg, 5])
    assert np.median(np.abs(rpg[bg, 5] - rp[bg, 5]) / np.abs(rp[bg, 5])) < 5e-3         # a few MeV of energy loss at most


def test_FFI_bookkeeping_every_root_is_fitted_single_tracks_too():
    tf, g, p, res, mr = _frame(1, 1)
    ok, ch, cp, rp, rc = oracle.refit_full(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev)
    n = len(ok)
    roots = mr.prev < 0
    singles = roots & (mr.next < 0)
    assert singles.sum() > 1000 and np.all(ok[roots] != 0) and (ok[singles] == 1).mean() > 0.97
    assert np.all(ok[~roots] == 0) and np.all(rc[~roots] == 0)
    np.testing.assert_array_equal(rp[~roots], res.tr_par[~roots])
    np.testing.assert_array_equal(rp[ok == -1], res.tr_par[ok == -1])
    assert np.all(rc[ok == -1] == 0)
    hits_by_root = np.bincount(mr.root, weights=res.tr_n_hits, minlength=n).astype(np.int64)
    np.testing.assert_array_equal(ch[roots], hits_by_root[roots])
    np.testing.assert_array_equal(cp[roots], np.bincount(mr.root, minlength=n)[roots])
    good = ok == 1
    # a covariance: positive diagonal, |correlation| <= 1
    d = rc[good][:, [0, 2, 5, 9, 14]]
    assert np.all(d > 0)
    for (a, b) in [(1, (1, 0)), (3, (2, 0)), (4, (2, 1)), (8, (3, 2)), (12, (4, 2)), (13, (4, 3))]:
        rho = rc[good, a] / np.sqrt(d[:, b[0]] * d[:, b[1]])
        assert np.all(np.abs(rho) <= 1.0 + 1e-3), a
    # the state sits on the innermost hit of the root piece
    r0 = (tf.row[res.tr_hit_index[res.tr_hit_offset[good]]].astype(np.int64)) % 152
    np.testing.assert_allclose(rp[good, 0], 85.0 + 1.07 * r0, atol=1e-4)
    assert np.all(rp[good, 6] == res.tr_par[good, 6])


# ---- FF-CE: chains that continue behind the central electrode (reading FF8) -------------------------------------------------

def test_FFCE_R_reflection_is_D_P_D_and_an_involution():
    rng = np.random.default_rng(2)
    L = rng.normal(size=(5, 5)) * np.array([0.2, 0.3, 0.02, 0.03, 0.4])[:, None]
    P0 = (L @ L.T).astype(np.float32).astype(np.float64)
    st0 = [120.0, 3.0, 7.25, 0.2, 0.375, -1.5]
    tc, tb, te = 5000.5, 4990.0, 4980.25                                        # all exact in fp32
    st, cv = oracle.full_reflect(st0, pack(P0), tc, tb, te)
    D = np.diag([1.0, -1.0, 1.0, -1.0, 1.0])
    assert np.array_equal(full(cv), (D @ P0 @ D).astype(np.float32).astype(np.float64))
    assert st[2] == np.float32(np.float32((2 * tc - tb - te)) * np.float32(0.516) - np.float32(7.25)) and st[4] == np.float32(-0.375)
    assert st[0] == 120.0 and st[1] == 3.0 and st[3] == np.float32(0.2) and st[5] == -1.5
    # the time of the point itself is mirrored about tc:  time' = 2 tc - time
    time_before = tb + 7.25 / 0.516
    assert abs((te + float(st[2]) / 0.516) - (2 * tc - time_before)) < 1e-3
    st2, cv2 = oracle.full_reflect(st, cv, tc, te, tb)                          # back again: the other side's reference first
    np.testing.assert_allclose(st2, np.array(st0, np.float32), atol=2e-3)
    assert np.array_equal(cv2, np.array(pack(P0), np.float32))


def _mirrored_line(slope=0.4, x_c=None, sec_a=3):
    """A straight line at y = 0 in sector sec_a (rows 60 .. 110, time rising outward with dz/dx = slope) that passes the electrode at
    x_c and goes on in the mirror sector (rows 112 .. 151, time falling with the same slope)."""
    from helpers import clusters_from_xyz, concat, row_x
    ra, rb = np.arange(60, 111), np.arange(112, 152)
    x_c = float(row_x(111)) if x_c is None else x_c
    z_c = 3000.0
    za = z_c - slope * (x_c - row_x(ra))
    zb = z_c - slope * (row_x(rb) - x_c)
    a = clusters_from_xyz(ra, np.zeros(ra.size), za, sector=sec_a)
    b = clusters_from_xyz(rb, np.zeros(rb.size), zb, sector=(sec_a + 18) % 36)
    return concat([a, b]), z_c / 0.516, ra, rb


def test_FFCE_L_mirrored_straight_line_is_fitted_as_one_line():
    """B = 0, y = 0: the two halves are ONE straight line in (x, reflected z).  After the refit across the electrode the state
    on the innermost hit has the true slope and z, and var(dz/ds) is that of a line fit through all 91 hits, not 51."""
    (row, pad, time), t_cross, ra, rb = _mirrored_line()
    g = oracle.default_geometry(36, 8000.0)
    p = oracle.default_params(0.08, 0.12)
    p.inv_R_per_qpt = 0.0
    res = oracle.track(g, p, row, pad, time)
    assert len(res.tr_seed) == 2 and sorted(res.tr_sector.tolist()) == [3, 21]
    mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
    ce = M.merge_ce(M.default_ce_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
    ia, ib = int(np.nonzero(res.tr_sector == 3)[0][0]), int(np.nonzero(res.tr_sector == 21)[0][0])
    assert mr.n_links == 0 and ce.n_links == 1 and ce.next[ia] == ib and abs(float(ce.t_ce[ia]) - t_cross) < 5e-3
    ok, ch, cp, rp, rc = oracle.refit_full_ce(g, p, row, pad, time, res, mr.next, mr.prev, ce.next, ce.prev, ce.t_ce, NO_MATERIAL)
    assert ok[ia] == 1 and ok[ib] == 0 and ch[ia] == ra.size + rb.size and cp[ia] == 2 and ch[ib] == rb.size
    np.testing.assert_array_equal(rp[ib], res.tr_par[ib])
    x60 = 85.0 + 1.07 * 60
    assert abs(rp[ia, 0] - x60) < 1e-4 and abs(rp[ia, 1]) < 1e-4 and abs(rp[ia, 3]) < 1e-5
    assert abs(rp[ia, 4] - 0.4) < 2e-4                                          # dz/ds of the A side, B's mirrored slope included
    z60 = (time[np.nonzero(row == 3 * 152 + 60)[0][0]] - rp[ia, 6]) * 0.516
    assert abs(rp[ia, 2] - z60) < 5e-3
    # var(t) of a straight-line fit: r_z / sum (x - mean x)^2 over ALL hits (the prior 1 / c0_t2 is negligible)
    xs = 85.0 + 1.07 * np.concatenate([ra, rb]).astype(np.float64)
    var_all = 0.12 ** 2 / np.sum((xs - xs.mean()) ** 2)
    var_a = 0.12 ** 2 / np.sum((xs[:ra.size] - xs[:ra.size].mean()) ** 2)
    assert abs(rc[ia, 9] / var_all - 1) < 0.02 and var_a > 4 * var_all, (rc[ia, 9], var_all, var_a)
    # without the C10 links the root is fitted from its own 51 hits
    ok0, ch0, _, rp0, rc0 = oracle.refit_full(g, p, row, pad, time, res, mr.next, mr.prev, NO_MATERIAL)
    assert ok0[ia] == 1 and ok0[ib] == 1 and ch0[ia] == ra.size and abs(rc0[ia, 9] / var_a - 1) < 0.02


def test_FFCE_H_noise_free_helices_and_FFCE_N_resolution_with_noise():
    import merge_eval as ME
    for noise_free in (True, False):
        c = gen.preset(1, 3)
        c.fixed_tracks, c.zv_sigma_cm, c.eta_max, c.pt_min = 3000, 30.0, 0.3, 0.3                 # many tracks through the electrode INSIDE the TPC
        if noise_free:
            c.sigma_y_cm = c.sigma_z_cm = c.dropout = c.noise_frac = 0.0
        tf = gen.generate(c)
        g, p = oracle.default_geometry(36, tf.max_time_bin), oracle.default_params()
        res = oracle.track(g, p, tf.row, tf.pad, tf.time)
        mr = M.merge(M.default_merge_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
        ce = M.merge_ce(M.default_ce_params(36), res.tr_seed, res.tr_sector, res.tr_first_row, res.tr_last_row, res.tr_par)
        ok0, ch0, cp0, rp0, rc0 = oracle.refit_full(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev, NO_MATERIAL)
        ok, ch, cp, rp, rc = oracle.refit_full_ce(g, p, tf.row, tf.pad, tf.time, res, mr.next, mr.prev, ce.next, ce.prev, ce.t_ce, NO_MATERIAL)
        used = np.array([a for a in np.nonzero(ce.next >= 0)[0] if mr.next[a] < 0 and mr.prev[ce.next[a]] < 0])
        assert used.size >= 250
        cont, roots = ce.next[used], mr.root[used]
        # bookkeeping: the continuation is no root any more, the root's chain holds both sides, everything else is plain C12
        assert np.all(ok[cont] == 0) and np.all(ok0[cont] == 1) and np.all(ok[roots] == 1)
        np.testing.assert_array_equal(rp[cont], res.tr_par[cont])
        pieces0 = np.bincount(mr.root, minlength=len(ok))
        hits0 = np.bincount(mr.root, weights=res.tr_n_hits, minlength=len(ok)).astype(np.int64)
        np.testing.assert_array_equal(cp[roots], pieces0[roots] + pieces0[cont])
        np.testing.assert_array_equal(ch[roots], hits0[roots] + hits0[cont])
        other = np.ones(len(ok), bool); other[roots] = False; other[cont] = False
        assert np.array_equal(ok[other], ok0[other]) and np.array_equal(rp[other], rp0[other]) and np.array_equal(rc[other], rc0[other])
        keys = ME.track_truth_keys(tf, res.tr_hit_offset, res.tr_n_hits, res.tr_hit_index)
        part = np.where(keys >= 0, keys // (64 * 16), 0)
        k_true = tf.tracks["charge_sense"][part] / tf.tracks["pt"][part]
        sel = roots[(keys[roots] >= 0) & ((keys[roots] % 16) % 2 == 0) & (ok0[roots] == 1)]
        assert sel.size >= 200
        h = res.tr_hit_index[res.tr_hit_offset[sel]]
        dz = np.abs(rp[sel, 2] - (tf.time[h] - rp[sel, 6]) * 0.516)
        dk, dk0 = np.abs(rp[sel, 5] - k_true[sel]), np.abs(rp0[sel, 5] - k_true[sel])
        assert np.mean(rc[sel, 14] < 0.5 * rc0[sel, 14]) > 0.9 and np.median(rc[sel, 14] / rc0[sel, 14]) < 0.05   # a much longer lever arm
        if noise_free:
            assert np.median(dz) < 1e-4 and np.quantile(dz, 0.95) < 0.05 and dz.max() < 0.6       # (a clamped crossing time shifts z by up to 2 * 0.5 bins)
            assert np.quantile(dk / np.abs(k_true[sel]), 0.95) < 1e-3
        else:
            assert np.median(dk) < 0.25 * np.median(dk0), (np.median(dk), np.median(dk0))
            pull = (rp[sel, 5] - k_true[sel]) / np.sqrt(rc[sel, 14])
            assert 0.8 < np.std(pull[np.abs(pull) < 8]) < 1.25
            assert np.median(dz) < 0.15


def test_FFCE_C_a_sector_boundary_link_takes_precedence_over_a_link_through_the_electrode():
    """FF8: the C10 link e -> b is used only if e has no C7 continuation and b is no C7 continuation of something else.
    Run with the three tracks in every order, so that track index 0 takes every role."""
    import itertools
    from helpers import clusters_from_xyz, concat, row_x
    (row, pad, time), t_cross, ra, rb = _mirrored_line()
    rc_ = np.arange(70, 115)
    c3 = clusters_from_xyz(rc_, np.full(rc_.size, 5.0), 900.0 + 0.2 * (row_x(rc_) - 85.0), sector=4)     # a third, unrelated track
    row, pad, time = concat([(row, pad, time), c3])
    g = oracle.default_geometry(36, 8000.0)
    p = oracle.default_params(0.08, 0.12)
    p.inv_R_per_qpt = 0.0
    res0 = oracle.track(g, p, row, pad, time)
    assert len(res0.tr_seed) == 3
    for order in itertools.permutations(range(3)):
        o = np.array(order)
        res = SimpleNamespace(tr_seed=res0.tr_seed[o], tr_sector=res0.tr_sector[o], tr_n_hits=res0.tr_n_hits[o], tr_hit_offset=res0.tr_hit_offset[o],
                              tr_hit_index=res0.tr_hit_index, tr_par=res0.tr_par[o])
        ia, ib, ic = (int(np.nonzero(res.tr_sector == s)[0][0]) for s in (3, 21, 4))
        none = np.full(3, -1, np.int32)
        ce_next, ce_prev, t_ce = none.copy(), none.copy(), np.zeros(3, np.float32)
        ce_next[ia], ce_prev[ib], t_ce[ia] = ib, ia, t_cross
        call = lambda nxt, prv: oracle.refit_full_ce(g, p, row, pad, time, res, nxt, prv, ce_next, ce_prev, t_ce, NO_MATERIAL)
        ok, ch, cp, _, _ = call(none, none)                                     # no conflict: A + B
        assert ok[ia] == 1 and ok[ib] == 0 and ok[ic] == 1 and ch[ia] == ra.size + rb.size and cp[ia] == 2 and ch[ic] == rc_.size, order
        nxt, prv = none.copy(), none.copy()
        nxt[ic], prv[ib] = ib, ic                                               # B already continues C across a sector boundary
        ok, ch, cp, _, _ = call(nxt, prv)
        assert ok[ia] == 1 and ch[ia] == ra.size and cp[ia] == 1, order         # A is fitted alone
        assert ok[ib] == 0 and ok[ic] != 0 and ch[ic] == rc_.size + rb.size and cp[ic] == 2, order
        nxt, prv = none.copy(), none.copy()
        nxt[ia], prv[ic] = ic, ia                                               # A already continues into C across a sector boundary
        ok, ch, cp, _, _ = call(nxt, prv)
        assert ok[ia] != 0 and ch[ia] == ra.size + rc_.size and cp[ia] == 2 and ok[ic] == 0, order
        assert ok[ib] == 1 and ch[ib] == rb.size and cp[ib] == 1, order         # B is a root of its own
