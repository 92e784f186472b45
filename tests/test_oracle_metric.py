"""Pins for the oracle's metric, derivatives, connection and acceleration.

None of these re-types an oracle formula: each compares the oracle with a mathematical fact
(an identity, a limit, a finite difference, another coordinate system).  CPU only.
"""
import numpy as np
import pytest

import closed_forms as cf
import oracle

RNG = np.random.default_rng(20170623)


def random_points(n, a, rmin=1.2, rmax=30.0):
    """Points outside the horizon, including the pole and the equator."""
    pts = []
    while len(pts) < n:
        p = RNG.uniform(-rmax, rmax, 3)
        if oracle.ks_r(a, *p) > rmin * cf.r_plus(a):
            pts.append(p)
    pts[0] = np.array([0.0, 0.0, 2.4])      # pole (Test C passes through it)
    pts[1] = np.array([2.9, -1.3, 0.0])     # equator
    return pts


@pytest.mark.parametrize("a", [0.0, 0.5, 0.9375, -0.99, 1.0])
def test_ks_radius_satisfies_eq5(a):
    # PAPER.md:65 eq. (5): x^2+y^2+z^2 = r^2 + a^2 (1 - z^2/r^2)
    for p in random_points(50, a):
        r = oracle.ks_r(a, *p)
        assert r > 0
        lhs = p @ p
        rhs = r * r + a * a * (1.0 - p[2] ** 2 / (r * r))
        assert abs(lhs - rhs) <= 1e-12 * lhs


@pytest.mark.parametrize("a", [0.0, 0.7, -0.9375, 1.0])
def test_l_is_unit_and_null_and_inverse(a):
    eta = np.diag([-1.0, 1.0, 1.0, 1.0])
    for p in random_points(30, a):
        g = oracle.ks_metric(a, p)
        gi = oracle.ks_metric_inverse(a, p)
        assert np.allclose(g, g.T, atol=1e-15, rtol=0)
        assert np.allclose(g @ gi, np.eye(4), atol=1e-12)
        # g - eta = f l l has rank one with l_0 = 1: recover f and l from g alone
        h = g - eta
        f = h[0, 0]
        l = h[0] / f
        assert abs(l[0] - 1.0) < 1e-14
        assert abs(l[1:] @ l[1:] - 1.0) < 1e-12          # spatial part is a unit vector
        assert abs(l @ np.linalg.inv(eta) @ l) < 1e-12   # null for eta
        assert abs(l @ gi @ l) < 1e-12                   # null for g
        assert np.allclose(h, f * np.outer(l, l), atol=1e-13)


def test_schwarzschild_limit():
    # a = 0: r = R, f = 2/r, l_i = x_i / r (ingoing Eddington-Finkelstein in Cartesian form)
    for p in random_points(20, 0.0):
        R = np.linalg.norm(p)
        assert abs(oracle.ks_r(0.0, *p) - R) < 1e-13 * R
        g = oracle.ks_metric(0.0, p)
        l = np.array([1.0, *(p / R)])
        expect = np.diag([-1.0, 1.0, 1.0, 1.0]) + (2.0 / R) * np.outer(l, l)
        assert np.allclose(g, expect, atol=1e-13)


@pytest.mark.parametrize("a", [0.5, 0.9375, -0.7])
def test_pullback_to_boyer_lindquist_is_eq1(a):
    # J^T g_KS J must equal the BL line element PAPER.md:47 eq. (1) (F11 replaces the missing Appendix)
    for _ in range(20):
        r = RNG.uniform(1.3 * cf.r_plus(a), 20.0)
        th = RNG.uniform(0.2, np.pi - 0.2)
        ph = RNG.uniform(0, 2 * np.pi)
        y, J = cf.bl_to_ks(a, (0.0, r, th, ph), np.zeros(4))
        g_ks = oracle.ks_metric(a, y[1:4])
        g_bl = oracle.bl_metric(a, [0.0, r, th, ph])
        # eq. (1) typed independently here
        rho2 = r * r + a * a * np.cos(th) ** 2
        delta = r * r - 2 * r + a * a
        s2 = np.sin(th) ** 2
        expect = np.zeros((4, 4))
        expect[0, 0] = -(1 - 2 * r / rho2)
        expect[0, 3] = expect[3, 0] = -2 * r * a * s2 / rho2
        expect[1, 1] = rho2 / delta
        expect[2, 2] = rho2
        expect[3, 3] = (r * r + a * a + 2 * r * a * a * s2 / rho2) * s2
        assert np.allclose(g_bl, expect, atol=1e-13)
        assert np.allclose(J.T @ g_ks @ J, expect, atol=1e-9 * max(1.0, np.abs(expect).max()))


@pytest.mark.parametrize("a", [0.0, 0.9, -0.9375, 1.0])
def test_analytic_dmetric_matches_central_differences(a):
    for p in random_points(25, a):
        dg = oracle.ks_dmetric(a, p)
        fd = oracle.ks_dmetric_fd(a, p, 1e-5)
        assert np.all(dg[0] == 0.0)                       # stationary
        assert np.allclose(dg, np.swapaxes(dg, 1, 2))     # symmetric in (a, b)
        assert np.allclose(dg, fd, atol=2e-9, rtol=1e-7)
        # and against a difference the test forms itself from oracle.ks_metric
        for c in range(3):
            e = np.zeros(3)
            e[c] = 1e-5
            mine = (oracle.ks_metric(a, p + e) - oracle.ks_metric(a, p - e)) / 2e-5
            assert np.allclose(dg[c + 1], mine, atol=2e-9, rtol=1e-7)


@pytest.mark.parametrize("a", [0.3, 0.99])
def test_christoffel_symmetry_and_metric_compatibility(a):
    for p in random_points(20, a):
        G = oracle.ks_christoffel(a, p)          # G[m, a, b]
        g = oracle.ks_metric(a, p)
        dg = oracle.ks_dmetric(a, p)             # dg[c, a, b]
        assert np.allclose(G, np.swapaxes(G, 1, 2), atol=1e-14)
        # nabla_c g_ab = 0  <=>  d_c g_ab = Gamma^d_ca g_db + Gamma^d_cb g_ad
        rhs = np.einsum("dca,db->cab", G, g) + np.einsum("dcb,ad->cab", G, g)
        assert np.allclose(dg, rhs, atol=1e-12)


def test_newtonian_limit():
    # slow particle far away: xdd^i -> -x_i / r^3
    for a in (0.0, 0.9):
        p = np.array([600.0, -500.0, 300.0])
        R = np.linalg.norm(p)
        acc = oracle.ks_accel(a, p, [1.0, 0.0, 0.0, 0.0])
        assert np.allclose(acc[1:], -p / R ** 3, rtol=2e-2)
        assert np.linalg.norm(acc[1:] + p / R ** 3) < 1e-2 * np.linalg.norm(p / R ** 3)


@pytest.mark.parametrize("a", [0.0, 0.8, -0.9375])
def test_accel_variants_agree(a):
    for p in random_points(15, a):
        u = RNG.uniform(-1, 1, 4)
        u[0] = 1.5
        an = oracle.ks_accel(a, p, u)
        fd = oracle.ks_accel_fd(a, p, u, 1e-5)
        assert np.allclose(an, fd, atol=1e-8, rtol=1e-7)
        # quadratic homogeneity of eq. (7)
        assert np.allclose(oracle.ks_accel(a, p, 2.0 * u), 4.0 * an, rtol=1e-13, atol=1e-15)


def solve_ut_by_sampling(a, kind, y):
    """Future-directed u^t with g u u = -mu^2: the norm is a quadratic in u^t; fit it from three samples."""
    n = []
    for ut in (0.0, 1.0, 2.0):
        yy = y.copy()
        yy[4] = ut
        n.append(oracle.invariants_one(a, kind, yy)[3] + (1.0 if kind == 1 else 0.0))
    C = n[0]
    A = (n[2] - 2.0 * n[1] + n[0]) / 2.0
    B = n[1] - n[0] - A
    roots = np.roots([A, B, C])
    return float(np.max(roots.real))


@pytest.mark.parametrize("a,kind", [(0.0, 0), (0.9, 0), (-0.9375, 1), (1.0, 0)])
def test_accel_conserves_all_four_invariants_instantaneously(a, kind):
    """A wrong sign, index or dropped term in Gamma breaks at least one of d/dlambda (norm, E, Lz, Q) = 0.
    The rate is formed by a centred difference of the invariants along (xd, xdd)."""
    eps = 1e-4
    for p in random_points(20, a, rmin=1.3):
        v = RNG.uniform(-0.6, 0.6, 3)
        y = np.array([0.0, *p, 2.0, *v])
        y[4] = solve_ut_by_sampling(a, kind, y)   # Q uses the nominal mu^2, so the state must have it
        acc = oracle.ks_accel(a, p, y[4:])
        dy = np.concatenate([y[4:], acc])
        d2 = np.concatenate([acc, np.zeros(4)])  # second-order position term keeps the difference O(eps^2)
        ip = oracle.invariants_one(a, kind, y + eps * dy + 0.5 * eps * eps * d2)
        im = oracle.invariants_one(a, kind, y - eps * dy + 0.5 * eps * eps * d2)
        rate = (ip - im) / (2 * eps)
        scale = np.abs(oracle.invariants_one(a, kind, y)) + np.array([1.0, 10.0, 100.0, 1.0])
        assert np.all(np.abs(rate) < 2e-6 * scale), (p, rate)
