"""Pins of the oracle's coordinate-time form (eq. 15).  CPU only.

The coordinate-time integrator is pinned against facts that do not depend on it: the chain rule that
links it to the affine form, the closed-form circular-orbit period in coordinate time, conserved
ratios, the paper's Table 1 altitude, the affine integration of the same geodesic (compared at equal
coordinate times), and 4th-order convergence."""
import numpy as np
import pytest

import closed_forms as cf
import oracle
from conftest import load_table1
from test_oracle_metric import random_points, solve_ut_by_sampling

RNG = np.random.default_rng(15)


@pytest.mark.parametrize("a", [0.0, 0.7, -0.9375])
def test_eq15_is_the_chain_rule_of_eq7(a):
    # v^i = u^i/u^t  =>  dv^i/dt = (xdd^i - v^i xdd^0) / (u^t)^2, and eq. (7) is quadratic in u
    for p in random_points(20, a, rmin=1.3):
        u = RNG.uniform(-0.7, 0.7, 4)
        u[0] = RNG.uniform(1.0, 3.0)
        acc = oracle.ks_accel(a, p, u)
        v = u[1:] / u[0]
        expect = (acc[1:] - v * acc[0]) / u[0] ** 2
        got = oracle.ks_coordtime_accel(a, p, v)
        assert np.allclose(got, expect, rtol=1e-12, atol=1e-15)


@pytest.mark.parametrize("a,r0,s", [(0.0, 8.0, +1), (0.7, 6.0, +1), (0.7, 10.0, -1)])
def test_circular_orbit_closes_after_one_coordinate_period(a, r0, s):
    omega, E, Lz, ut = cf.circular_orbit(a, r0, s)
    st = cf.ks_state_on_equator(a, r0, ut, omega * ut, 0.0)
    y0 = np.array([0.0, *st[1:4], *(st[5:8] / st[4])])
    T = 2 * np.pi / abs(omega)
    n = 4096
    traj = oracle.trajectory_coordtime(a, y0, T / n, n, stride=n // 8)
    r = np.array([oracle.ks_r(a, *row[1:4]) for row in traj])
    assert np.abs(r - r0).max() < 1e-9
    assert abs(traj[-1, 0] - T) < 1e-9 and np.abs(traj[-1, 1:4] - y0[1:4]).max() < 1e-8
    # |v| = r Omega in the orbital plane, constant
    assert np.allclose(np.linalg.norm(traj[:, 4:7], axis=1), np.linalg.norm(y0[4:7]), rtol=1e-10)


@pytest.mark.parametrize("kind,a", [(0, 0.9), (1, 0.6), (0, -0.5)])
def test_conserved_ratios_along_a_coordinate_time_trajectory(kind, a):
    # with v^0 = 1 the tangent is u/u^t: xi = Lz/E and eta = Q/E^2 (null), E/sqrt(-u.u) (time-like) are constant
    pos = np.array([9.0, -2.0, 3.0])
    y8 = np.array([0.0, *pos, 1.0, -0.35, 0.6, 0.15]) if kind == 0 else np.array([0.0, *pos, 1.0, 0.05, 0.28, 0.08])
    y8[4] = solve_ut_by_sampling(a, kind, y8)
    y0 = np.array([0.0, *pos, *(y8[5:8] / y8[4])])
    traj = oracle.trajectory_coordtime(a, y0, 0.02, 3000, stride=300)
    vals = []
    for row in traj:
        E, Lz, Q, norm = oracle.invariants_one(a, 0, np.array([row[0], *row[1:4], 1.0, *row[4:7]]))
        c = row[3] / oracle.ks_r(a, *row[1:4])
        Q = Q + a * a * c * c * (-norm)        # Carter's constant with mu^2 = -u.u of this tangent (not the nominal 0)
        vals.append([Lz / E, Q / E ** 2, norm / E ** 2])
    vals = np.array(vals)
    assert np.abs(vals - vals[0]).max() < 2e-7, np.abs(vals - vals[0]).max(axis=0)
    if kind == 0:
        assert np.abs(vals[:, 2]).max() < 1e-8      # stays null


def _hermite(t0, x0, v0, t1, x1, v1, t):
    h = t1 - t0
    s = (t - t0) / h
    return ((2 * s ** 3 - 3 * s ** 2 + 1) * x0 + (s ** 3 - 2 * s ** 2 + s) * h * v0 +
            (-2 * s ** 3 + 3 * s ** 2) * x1 + (s ** 3 - s ** 2) * h * v1)


@pytest.mark.parametrize("case", range(4))
def test_same_curve_as_the_affine_integration_at_equal_times(case):
    a = [0.9, 0.0, -0.7, 0.5][case]
    kind = case % 2
    pos = np.array([[12.0, 3.0, -2.0], [8.0, -6.0, 1.0], [0.5, 10.0, 4.0], [-9.0, 2.0, 6.0]][case])
    vel = np.array([[-0.9, 0.25, 0.1], [-0.2, 0.3, 0.05], [0.3, -0.8, -0.2], [0.4, 0.1, -0.3]][case])
    y8 = np.array([0.0, *pos, 1.0, *vel])
    y8[4] = solve_ut_by_sampling(a, kind, y8)
    aff = oracle.trajectory(a, y8, 1.0 / 256, 256 * 20)              # fine affine run: rows t,x,y,z,u
    y0 = np.array([0.0, *pos, *(vel / y8[4])])
    errs = []
    for dt in (0.1, 0.05):
        n = int(round(12.0 / dt))
        ct = oracle.trajectory_coordtime(a, y0, dt, n, stride=n // 6)
        e = 0.0
        for row in ct[1:]:
            k = np.searchsorted(aff[:, 0], row[0]) - 1
            assert 0 <= k < len(aff) - 1
            x = _hermite(aff[k, 0], aff[k, 1:4], aff[k, 5:8] / aff[k, 4], aff[k + 1, 0], aff[k + 1, 1:4],
                         aff[k + 1, 5:8] / aff[k + 1, 4], row[0])
            e = max(e, np.abs(x - row[1:4]).max())
        errs.append(e)
    assert errs[1] < 2e-6, errs
    assert errs[0] / errs[1] > 8.0 or errs[0] < 1e-9, errs      # 4th order in dt


def test_table1_altitude_in_coordinate_time():
    # Test B of Table 1 integrated with respect to t reaches the same max|cos theta|
    row = load_table1()[1]
    y8, phi, q = cf.spherical_photon_state(1.0, row["r"])
    y0 = np.array([0.0, *y8[1:4], *(y8[5:8] / y8[4])])
    traj = oracle.trajectory_coordtime(1.0, y0, 0.01, 4000)
    r = np.array([oracle.ks_r(1.0, *p) for p in traj[:, 1:4]])
    c = np.abs(traj[:, 3] / r)
    i = 1
    while not (c[i] >= c[i - 1] and c[i] > c[i + 1]):
        i += 1
    peak = c[i] - (c[i + 1] - c[i - 1]) ** 2 / (8.0 * (c[i - 1] - 2 * c[i] + c[i + 1]))
    assert abs(peak - row["maxcos"]) < 6e-5 and np.abs(r[: i + 1] - row["r"]).max() < 1e-6


def test_driver_stops_at_the_target_time_and_resumes():
    xu8 = np.array([cf.circular_orbit_state(0.7, 9.0, +1), cf.circular_orbit_state(0.7, 14.0, -1)])
    st = oracle.init_timelike(0.7, xu8)
    sc = oracle.step_control(mode=0, h_fixed=0.7, max_steps=100000)
    s1 = oracle.integrate_coordtime(st, 100.0, sc)
    assert (st.status == oracle.ACTIVE).all() and np.allclose(st.q[0], 100.0, atol=1e-12)
    assert (st.nsteps == 143).all() and s1["steps"] == 286            # 142 full steps + one clipped
    assert np.allclose(st.q[4], 1.0)
    one = oracle.init_timelike(0.7, xu8)
    oracle.integrate_coordtime(one, 250.0, sc)
    oracle.integrate_coordtime(st, 250.0, sc)
    assert np.allclose(one.q[1:4], st.q[1:4], atol=1e-6) and np.allclose(st.q[0], 250.0, atol=1e-12)
    r = [oracle.ks_r(0.7, *st.q[1:4, k]) for k in range(2)]
    assert np.allclose(r, [9.0, 14.0], atol=1e-6)
    again = oracle.integrate_coordtime(st, 250.0, sc)
    assert again["steps"] == 0
    # capture / escape tests run on t-steps too
    img = oracle.init_null(0.5, 60.0, np.radians(45.0), 8.0, 8.0, 6, 6)
    stats = oracle.integrate_coordtime(img, float("inf"), oracle.step_control(mode=1, eta=0.02, r_escape=70.0))
    assert stats["n_active"] == 0 and stats["n_captured"] > 0 and stats["n_escaped"] > 0
    ref = oracle.init_null(0.5, 60.0, np.radians(45.0), 8.0, 8.0, 6, 6)
    oracle.integrate(ref, float("inf"), oracle.step_control(mode=1, eta=0.02, r_escape=70.0))
    assert np.array_equal(ref.status, img.status)      # same geodesics, same fate
