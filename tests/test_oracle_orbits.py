"""Pins of the oracle integrator against GR textbook facts for orbits, the independent
Boyer-Lindquist integration, and the driver-loop semantics.  CPU only."""
import numpy as np
import pytest

import closed_forms as cf
import oracle
from conftest import load_table1
from paper_1706_07062_b200 import inputs

INF = float("inf")


def radius(a, traj):
    return np.array([oracle.ks_r(a, *p) for p in traj[:, 1:4]])


# ---- Schwarzschild photon sphere ------------------------------------------------------------------

def test_schwarzschild_photon_sphere_at_3M():
    # PAPER.md:194-197 with a = 0: r_p = r_r = 3M.  Tangential photon at r = 3 with L/E = sqrt(27).
    assert abs(cf.r_photon_prograde(0.0) - 3.0) < 1e-12 and abs(cf.r_photon_retrograde(0.0) - 3.0) < 1e-12
    b = np.sqrt(27.0)
    # E = (1 - 2/r) u^t = 1 -> u^t = 3 ; u^phi = L / r^2 = b / 9 ; tangential velocity r u^phi = b / 3
    y0 = np.array([0.0, 3.0, 0.0, 0.0, 3.0, 0.0, b / 3.0, 0.0])
    E, Lz, Q, norm = oracle.invariants_one(0.0, 0, y0)
    assert abs(E - 1) < 1e-14 and abs(Lz - b) < 1e-14 and abs(norm) < 1e-14
    traj = oracle.trajectory(0.0, y0, 1.0 / 64, 64 * 30, stride=64)
    dr = np.abs(radius(0.0, traj) - 3.0)
    assert dr[:13].max() < 1e-6        # one full revolution takes lambda = 2 pi r^2 / L = 10.9
    # unstable: delta r grows as exp(kappa lambda), kappa^2 = -V''/2 = 1/3 for V = (1-2/r) L^2/r^2 at r = 3
    growth = np.log(dr[-1] / dr[-6]) / 5.0
    assert abs(growth - 1.0 / np.sqrt(3.0)) < 0.01
    # slightly inside / outside: falls in / flies out (instability separates capture from escape)
    for eps, expect in ((-1e-3, oracle.CAPTURED), (+1e-3, oracle.ESCAPED)):
        y = y0.copy()
        y[1] += eps
        st = oracle.init_explicit(0.0, y[None, :], oracle.NULL)
        oracle.integrate(st, INF, oracle.step_control(mode=0, h_fixed=1.0 / 32, r_escape=50.0, max_steps=200000))
        assert st.status[0] == expect


# ---- circular time-like orbits: period, constancy of r, E and Lz (F8) -----------------------------

@pytest.mark.parametrize("a,r0,s", [(0.0, 8.0, +1), (0.7, 6.0, +1), (0.7, 10.0, -1), (-0.7, 10.0, +1)])
def test_circular_orbit_period_and_constants(a, r0, s):
    omega, E, Lz, ut = cf.circular_orbit(abs(a), r0, s if a >= 0 else -s)
    if a < 0:  # Kerr(-a) is the mirror image: same orbit with phi -> -phi
        omega, Lz = -omega, -Lz
    st = cf.ks_state_on_equator(a, r0, ut, omega * ut, 0.0)
    inv = oracle.invariants_one(a, oracle.TIMELIKE, st)
    assert np.allclose(inv, [E, Lz, 0.0, -1.0], atol=1e-12)
    if a == 0.0:
        assert abs(2 * np.pi / abs(omega) - 2 * np.pi * r0 ** 1.5) < 1e-12
    # integrate exactly one coordinate-time period T = 2 pi / |Omega| : dt/dlambda = u^t is constant
    lam_T = 2 * np.pi / abs(omega) / ut
    n = 4096
    traj = oracle.trajectory(a, st, lam_T / n, n, stride=n // 64)
    assert np.abs(radius(a, traj) - r0).max() < 1e-9
    assert abs(traj[-1, 0] - 2 * np.pi / abs(omega)) < 1e-8
    assert np.abs(traj[-1, 1:4] - st[1:4]).max() < 1e-8        # phi closes after T
    # and a quarter period is a quarter turn in the right direction
    q = traj[16]
    ang = np.arctan2(q[2], q[1]) - np.arctan2(st[2], st[1])
    assert abs((ang - np.sign(omega) * np.pi / 2 + np.pi) % (2 * np.pi) - np.pi) < 1e-8


# ---- ISCO (F9) ------------------------------------------------------------------------------------

def test_isco_radii_closed_form_values():
    assert abs(cf.r_isco(0.0) - 6.0) < 1e-12
    assert abs(cf.r_isco(0.7, +1) - 3.39313) < 1e-5 and abs(cf.r_isco(0.7, -1) - 8.14297) < 1e-5
    assert abs(cf.r_isco(0.9375, +1) - 2.04420) < 1e-5


@pytest.mark.parametrize("a,s", [(0.0, +1), (0.7, +1), (0.7, -1), (0.9375, +1)])
def test_isco_separates_stable_from_plunging(a, s):
    """A circular orbit nudged inward (u^x-kick of -1e-4 along the radial direction) oscillates when
    outside r_isco and plunges to the horizon when inside."""
    risco = cf.r_isco(a, s)
    results = {}
    for tag, r0 in (("stable", 1.10 * risco), ("unstable", 0.90 * risco)):
        st = cf.circular_orbit_state(a, r0, s)
        x, y = st[1], st[2]
        nrm = np.hypot(x, y)
        st[5] -= 1e-4 * x / nrm
        st[6] -= 1e-4 * y / nrm
        state = oracle.init_timelike(a, st[None, :], renormalise_ut=True)
        T = 2 * np.pi * (r0 ** 1.5 + s * a)
        sc = oracle.step_control(mode=0, h_fixed=0.05, r_escape=INF, max_steps=int(40 * T / 0.05))
        oracle.integrate(state, INF, sc)
        results[tag] = (state.status[0], oracle.ks_r(a, *state.q[1:4, 0]))
    assert results["stable"][0] == oracle.MAXSTEPS and abs(results["stable"][1] - 1.10 * risco) < 0.05 * risco
    assert results["unstable"][0] == oracle.CAPTURED


# ---- vertical epicyclic frequency (F10; Fig. 9) ---------------------------------

@pytest.mark.parametrize("a,r0", [(1.0, 1.4), (1.0, 4.0), (0.9, 4.0), (0.0, 8.0)])
def test_vertical_epicyclic_frequency(a, r0):
    # the paper's recipe: v_z = 1e-12 kick, linear interpolation in z(t), time between successive maxima
    st = cf.circular_orbit_state(a, r0, +1, vz=1e-12)
    expect = cf.vertical_epicyclic(a, r0, +1)
    omega, _, _, ut = cf.circular_orbit(a, r0, +1)
    T_perp = 2 * np.pi / expect
    h = T_perp / ut / 2048.0
    traj = oracle.trajectory(a, st, h, int(2.6 * 2048))
    t, z = traj[:, 0], traj[:, 3]
    # maxima of z <=> downward zero crossings of u^z, located by linear interpolation in t
    uz = traj[:, 7]
    cross = [k for k in range(len(uz) - 1) if uz[k] > 0.0 >= uz[k + 1]]
    tm = [t[k] + (t[k + 1] - t[k]) * uz[k] / (uz[k] - uz[k + 1]) for k in cross[:2]]
    assert len(tm) == 2
    measured = 2 * np.pi / (tm[1] - tm[0])
    assert abs(measured / expect - 1.0) < 1e-7, (measured, expect)
    assert np.abs(z).max() < 1e-10   # stays a tiny perturbation


# ---- independent Boyer-Lindquist integration of the same geodesics (C8) ---------------------------

def _bl_initial_from_ks(a, y_ks):
    """Convert a KS Cartesian state to BL using the F11 map and its Jacobian (closed_forms)."""
    r, th, ph = cf.ks_to_bl_position(a, y_ks[1:4])
    y_back, J = cf.bl_to_ks(a, (0.0, r, th, ph), np.zeros(4))
    assert np.allclose(y_back[1:4], y_ks[1:4], atol=1e-11)
    u_bl = np.linalg.solve(J, y_ks[4:])
    return np.array([0.0, r, th, ph, *u_bl]), y_back[0]


@pytest.mark.parametrize("case", range(6))
def test_boyer_lindquist_cross_integration(case):
    rng = np.random.default_rng(100 + case)
    a = [0.5, 0.9, -0.7, 0.0, 0.9375, 0.3][case]
    kind = case % 2
    # start away from the poles and the horizon with a moderately inclined velocity
    r0 = rng.uniform(5.0, 9.0)
    th0 = rng.uniform(1.1, 2.0)
    ph0 = rng.uniform(0, 2 * np.pi)
    y, J = cf.bl_to_ks(a, (0.0, r0, th0, ph0), np.zeros(4))
    vdir = rng.normal(size=3)
    vdir /= np.linalg.norm(vdir)
    speed = 1.0 if kind == 0 else 0.35
    y[5:8] = speed * vdir
    st = oracle.init_timelike(a, y[None, :], renormalise_ut=True) if kind == 1 else None
    if kind == 0:
        # null: solve u^t by sampling the norm (a quadratic in u^t)
        from test_oracle_metric import solve_ut_by_sampling
        y[4] = solve_ut_by_sampling(a, 0, y)
    else:
        y[4] = st.q[4, 0]
    y_bl, t_shift = _bl_initial_from_ks(a, y)
    errs = []
    for n in (64, 128):
        nsteps = 6 * n
        tk = oracle.trajectory(a, y, 1.0 / n, nsteps, stride=n)
        tb = oracle.bl_trajectory(a, y_bl, 1.0 / n, nsteps, stride=n)
        rk = radius(a, tk)
        assert rk.min() > 1.2 * cf.r_plus(a)
        thk = np.arccos(tk[:, 3] / rk)
        assert np.abs(np.cos(thk)).max() < 0.95
        e_r = np.abs(rk - tb[:, 1]).max()
        e_th = np.abs(thk - tb[:, 2]).max()
        phk = np.array([cf.ks_to_bl_position(a, p)[2] for p in tk[:, 1:4]])
        e_ph = np.abs((phk - tb[:, 3] + np.pi) % (2 * np.pi) - np.pi).max()
        errs.append(max(e_r, e_th, e_ph))
    assert errs[1] < 2e-8, errs
    assert errs[0] / errs[1] > 6.0 or errs[0] < 1e-10, errs   # shrinks ~16x per halving (two RK4 truncations)


# ---- driver loop semantics (C5) -------------------------------------------------------------------

def _one_ray(a=0.5):
    st = oracle.init_null(a, 50.0, np.radians(60.0), 8.0, 8.0, 4, 4)
    return st


def test_resume_equals_one_shot_and_second_call_is_noop():
    sc = oracle.step_control(mode=1, eta=0.02, r_escape=60.0, max_steps=5000)
    one = _one_ray()
    oracle.integrate(one, 45.0, sc)
    two = _one_ray()
    oracle.integrate(two, 30.0, sc)
    assert (two.status == oracle.ACTIVE).all() and np.allclose(two.lam, 30.0, atol=1e-12)
    oracle.integrate(two, 45.0, sc)
    both = (one.status == oracle.ACTIVE) & (two.status == oracle.ACTIVE)
    assert both.sum() >= 8 and np.allclose(one.lam[both], 45.0, atol=1e-12) and np.allclose(two.lam[both], 45.0, atol=1e-12)
    # the clipped step changes the step sequence, so states agree to truncation level only
    assert np.allclose(one.q[1:4][:, both], two.q[1:4][:, both], rtol=0, atol=1e-3)
    d = two.nsteps[both] - one.nsteps[both]
    assert ((d == 0) | (d == 1)).all()   # at most one extra (clipped) step at lambda = 30
    oracle.integrate(one, INF, sc)
    oracle.integrate(two, INF, sc)
    assert (one.status == two.status).all() and (one.status != oracle.ACTIVE).all()
    before = two.copy()
    stats = oracle.integrate(two, INF, sc)
    assert stats["steps"] == 0 and np.array_equal(before.q, two.q) and np.array_equal(before.nsteps, two.nsteps)


def test_max_steps_is_exact_and_absolute():
    xu8 = cf.circular_orbit_state(0.7, 9.0, +1)[None, :]
    st = oracle.init_timelike(0.7, xu8)
    sc = oracle.step_control(mode=0, h_fixed=0.5, max_steps=100)
    s1 = oracle.integrate(st, INF, sc)
    assert s1["steps"] == 100 and st.status[0] == oracle.MAXSTEPS and st.nsteps[0] == 100
    assert abs(st.lam[0] - 50.0) < 1e-12
    st.status[0] = oracle.ACTIVE
    s2 = oracle.integrate(st, INF, oracle.step_control(mode=0, h_fixed=0.5, max_steps=150))
    assert s2["steps"] == 50 and st.nsteps[0] == 150


def test_status_codes_and_invalid_input():
    st = oracle.init_null(0.0, 100.0, np.radians(60.0), 10.0, 10.0, 8, 8)
    st.q[5, 3] = np.nan
    sc = oracle.step_control(mode=1, eta=0.01, r_escape=150.0, max_steps=20000)
    stats = oracle.integrate(st, INF, sc)
    assert st.status[3] == oracle.INVALID and st.nsteps[3] == 0
    assert stats["n_invalid"] == 1 and stats["n_active"] == 0
    assert stats["n_captured"] + stats["n_escaped"] == 63
    assert stats["steps"] == int(st.nsteps.sum())
    # final state is the state at which the test fired: captured rays sit just inside 1.01 r_plus
    r = np.array([oracle.ks_r(0.0, *st.q[1:4, k]) for k in range(64)])
    cap = st.status == oracle.CAPTURED
    assert cap.any() and (r[cap] < 1.01 * 2.0).all() and (r[cap] > 0.9 * 2.0).all()
    esc = st.status == oracle.ESCAPED
    assert (r[esc] > 150.0).all() and (r[esc] < 150.0 * 1.02).all()


def test_backward_direction_runs_time_reversed():
    # dir = -1 with the same state retraces a forward segment (time-like, far from the hole)
    xu8 = cf.circular_orbit_state(0.3, 12.0, +1)[None, :]
    st = oracle.init_timelike(0.3, xu8)
    fwd = oracle.step_control(mode=0, h_fixed=0.25, max_steps=1000)
    oracle.integrate(st, 100.0, fwd)
    assert abs(st.lam[0] - 100.0) < 1e-12 and st.status[0] == oracle.ACTIVE
    bwd = oracle.step_control(mode=0, h_fixed=0.25, dir=-1, max_steps=2000)
    oracle.integrate(st, 0.0, bwd)
    assert abs(st.lam[0]) < 1e-12
    assert np.allclose(st.q[:, 0], xu8[0], atol=1e-7)


def test_renormalise_ut_gives_unit_norm():
    rng = np.random.default_rng(3)
    xu8 = np.zeros((10, 8))
    xu8[:, 1:4] = rng.uniform(4, 12, (10, 3))
    xu8[:, 5:8] = rng.uniform(-0.3, 0.3, (10, 3))
    xu8[:, 4] = 123.0
    st = oracle.init_timelike(0.8, xu8, renormalise_ut=True)
    assert np.abs(oracle.invariants(st)[3] + 1.0).max() < 1e-13 and (st.q[4] > 0).all()
    raw = oracle.init_timelike(0.8, xu8, renormalise_ut=False)
    assert np.array_equal(raw.q[4], xu8[:, 4])


# ---- equatorial circular photon orbits, eq. (19)-(20) ----------------------------

@pytest.mark.parametrize("a", [0.5, 0.9])
def test_circular_photon_orbit_radii_of_eq19_eq20(a):
    rp, rr = cf.r_photon_prograde(a), cf.r_photon_retrograde(a)
    assert 1.0 <= rp <= 3.0 <= rr <= 4.0                               # the inequality below eq. (20)
    for r0, sign in ((rp, +1), (rr, -1)):
        phi, q = cf.teo_phi_q(a, r0)
        assert abs(q) < 1e-9 and np.sign(phi) == sign                   # equatorial (Q = 0), pro-/retrograde
        y0, _, _ = cf.spherical_photon_state(a, r0)
        y0[7] = 0.0                                                     # Q = 0 up to rounding: stay in the plane
        traj = oracle.trajectory(a, y0, 1.0 / 512, 512 * 6, stride=64)
        assert np.abs(radius(a, traj) - r0).max() < 1e-6                # circular (unstable: truncation error grows)
        assert np.abs(traj[:, 3]).max() < 1e-12
        ang = np.unwrap(np.arctan2(traj[:, 2], traj[:, 1]))
        assert np.sign(ang[-1] - ang[0]) == sign
        # a photon slightly outside r_r escapes, slightly inside r_p is captured (same constants of motion)
    for r0, eps, expect in ((rr, +2e-3, oracle.ESCAPED), (rp, -2e-3, oracle.CAPTURED)):
        y0, _, _ = cf.spherical_photon_state(a, r0)
        y0[7] = 0.0
        scale = (r0 + eps) / r0
        y0[1] *= scale
        y0[2] *= scale
        st = oracle.init_explicit(a, y0[None, :], oracle.NULL)
        oracle.integrate(st, INF, oracle.step_control(mode=0, h_fixed=1.0 / 64, r_escape=40.0, max_steps=400000))
        assert st.status[0] == expect


# ---- explicit initial data of either kind (Table 1: photons; particles) -----

def test_init_explicit_records_the_kind_and_uses_it():
    """Table 1's spherical photon orbits are explicit NULL data: the state-level invariants must return the
    paper's (Phi, Q) with mu^2 = 0; declared TIMELIKE the same 8-vector has Q lower by a^2 cos^2(theta) = 0 on
    the equator but its re-solved u^t differs (g u u = -1 instead of 0)."""
    a, row = 1.0, load_table1()[4]                    # row E, outside the ergosphere: 1 - f > 0
    y0, phi, q = cf.spherical_photon_state(a, row["r"])
    st = oracle.init_explicit(a, y0[None, :], oracle.NULL)
    assert (st.kind, st.reversed, st.a_eff) == (oracle.NULL, 0, a)
    E, Lz, Q, norm = oracle.invariants(st)
    assert abs(E[0] - 1) < 1e-13 and abs(Lz[0] - row["phi"]) < 5e-5 and abs(Q[0] - row["q"]) < 5e-5 and abs(norm[0]) < 1e-13
    # off the equator mu^2 enters Q: a^2 cos^2(theta) (mu^2 - E^2)
    tr = oracle.trajectory(a, y0, 1.0 / 64, 64)[-1]
    Qn = oracle.invariants(oracle.init_explicit(a, tr[None, :], oracle.NULL))[2][0]
    Qt = oracle.invariants(oracle.init_explicit(a, tr[None, :], oracle.TIMELIKE))[2][0]
    c2 = (tr[3] / oracle.ks_r(a, *tr[1:4])) ** 2
    assert abs((Qt - Qn) - a * a * c2) < 1e-12 and c2 > 0.01
    # u^t re-solved from g u u = -mu^2
    bad = y0.copy(); bad[4] = 99.0
    n0 = oracle.invariants(oracle.init_explicit(a, bad[None, :], oracle.NULL, renormalise_ut=True))[3][0]
    n1 = oracle.invariants(oracle.init_explicit(a, bad[None, :], oracle.TIMELIKE, renormalise_ut=True))[3][0]
    assert abs(n0) < 1e-13 and abs(n1 + 1.0) < 1e-13
    assert abs(oracle.init_explicit(a, bad[None, :], oracle.NULL, renormalise_ut=True).q[4, 0] - y0[4]) < 1e-12
    # init_timelike is the TIMELIKE case
    t = oracle.init_timelike(a, bad[None, :], renormalise_ut=True)
    e = oracle.init_explicit(a, bad[None, :], oracle.TIMELIKE, renormalise_ut=True)
    assert t.kind == oracle.TIMELIKE and np.array_equal(t.q, e.q)


def test_clipped_last_step_lands_on_lambda_end_exactly():
    """DESIGN R22: the clipped step ends at lambda_end itself.  In double 0.03 + (0.283 - 0.03) > 0.283 and
    0.05 + (0.216 - 0.05) < 0.216, so a clock advanced by lambda += h would overshoot by an ulp in the first
    case and stop an ulp short -- and take one more, ulp-sized, step -- in the second."""
    assert 0.03 + (0.283 - 0.03) > 0.283 and 0.05 + (0.216 - 0.05) < 0.216
    xu8, _ = inputs.cfg1_orbits(4)
    for driver in (oracle.integrate, oracle.integrate_coordtime):
        for first, second in ((0.03, 0.283), (0.05, 0.216)):
            st = oracle.init_timelike(0.0, xu8)
            sc = oracle.step_control(mode=0, h_fixed=1.0, max_steps=10 ** 6)
            assert driver(st, first, sc)["steps"] == 4
            stats = driver(st, second, sc)
            clock = st.lam if driver is oracle.integrate else st.q[0]
            assert (clock == second).all() and stats["steps"] == 4 and (st.status == oracle.ACTIVE).all()
            assert driver(st, second, sc)["steps"] == 0               # a second identical call is a no-op
