"""The seeded input generators: determinism, the stated distributions, and physical validity of
what they produce (checked through the oracle's invariants and a short oracle integration).  CPU only."""
import numpy as np

import closed_forms as cf
import oracle
from paper_1706_07062_b200 import inputs


def test_splitmix64_reference_values_and_determinism():
    # first outputs of the published splitmix64 generator for seed 0 (state advances by the golden gamma)
    u = inputs.splitmix64_uniform(0, np.arange(3))
    z0 = 0xE220A8397B1DCDAF
    assert abs(u[0] - (z0 >> 11) / 2.0 ** 53) == 0.0
    assert np.array_equal(u, inputs.splitmix64_uniform(0, np.arange(3)))
    big = inputs.splitmix64_uniform(7062, np.arange(200000))
    assert 0.0 <= big.min() and big.max() < 1.0
    assert abs(big.mean() - 0.5) < 5e-3 and abs(big.var() - 1.0 / 12.0) < 2e-3


def test_cfg1_orbits_are_circular_geodesics():
    xu8, r0 = inputs.cfg1_orbits()
    assert xu8.shape == (16, 8) and ((r0 > 6.0) & (r0 <= 20.0)).all()
    st = oracle.init_timelike(0.0, xu8)
    E, Lz, Q, norm = oracle.invariants(st)
    assert np.abs(norm + 1.0).max() < 1e-13
    # Schwarzschild circular orbit: E = (1-2/r)/sqrt(1-3/r), L^2 = Lz^2 + Q = r^2/(r-3)
    assert np.allclose(E, (1 - 2 / r0) / np.sqrt(1 - 3 / r0), atol=1e-13)
    assert np.allclose(Lz ** 2 + Q, r0 ** 2 / (r0 - 3.0), rtol=1e-12)
    sc = oracle.step_control(mode=0, h_fixed=0.5, max_steps=5000)
    oracle.integrate(st, float("inf"), sc)
    r = np.array([oracle.ks_r(0.0, *st.q[1:4, k]) for k in range(16)])
    assert (st.status == oracle.MAXSTEPS).all() and (st.nsteps == 5000).all()
    assert np.abs(r - r0).max() < 1e-3            # r constant to O(h^4); worst is r0 = 6.48, close to the ISCO
    again, _ = inputs.cfg1_orbits()
    assert np.array_equal(xu8, again)


def test_cfg4_ensemble_is_bound_and_matches_solved_constants():
    n = 2048
    xu8, meta = inputs.cfg4_ensemble(n)
    xu8b, _ = inputs.cfg4_ensemble(n)
    assert np.array_equal(xu8, xu8b)
    assert 0.95 < meta["acceptance"] <= 1.0
    assert (meta["p"] >= 8).all() and (meta["p"] <= 50).all() and (meta["e"] >= 0).all() and (meta["e"] <= 0.8).all()
    assert abs(meta["cosi"].mean()) < 0.1 and (np.abs(meta["cosi"]) <= 1).all()
    st = oracle.init_timelike(0.7, xu8)
    E, Lz, Q, norm = oracle.invariants(st)
    assert np.abs(E - meta["E"]).max() < 1e-13 and np.abs(Lz - meta["Lz"]).max() < 1e-12
    assert np.abs(Q - meta["Q"]).max() < 1e-11 and np.abs(norm + 1.0).max() < 1e-12
    assert (E < 1.0).all()
    # cos iota = Lz / sqrt(Lz^2 + Q)
    assert np.allclose(Lz / np.sqrt(Lz ** 2 + Q), meta["cosi"], atol=1e-12)
    # starts at apoapsis on the equator
    ra = meta["p"] / (1 - meta["e"])
    r_start = np.array([oracle.ks_r(0.7, *xu8[k, 1:4]) for k in range(n)])
    assert np.allclose(r_start, ra, rtol=1e-13) and (xu8[:, 3] == 0).all()


def test_cfg4_orbits_stay_between_their_turning_points():
    xu8, meta = inputs.cfg4_ensemble(64)
    rp, ra = meta["p"] / (1 + meta["e"]), meta["p"] / (1 - meta["e"])
    rmin = np.full(64, np.inf)
    rmax = np.zeros(64)
    for k in range(64):
        traj = oracle.trajectory(0.7, xu8[k], 0.5, 6000, stride=4)
        r = np.array([oracle.ks_r(0.7, *p) for p in traj[:, 1:4]])
        rmin[k], rmax[k] = r.min(), r.max()
    assert (rmax <= ra * (1 + 1e-6)).all() and (rmin >= rp * (1 - 1e-3)).all()
    # orbits with short periods have reached periapsis within 3000 M of affine parameter
    short = ra < 40
    assert (rmin[short] < rp[short] * 1.05).all()


def test_cfg4_generator_newton_matches_circular_closed_form():
    # e = 0, equatorial: must reproduce the Bardeen-Press-Teukolsky circular orbit constants
    for s, c in ((+1, 1.0), (-1, -1.0)):
        E, Lz, Q, ok = inputs.solve_orbit_constants(0.7, np.array([12.0]), np.array([0.0]), np.array([c]))
        _, Ec, Lc, _ = cf.circular_orbit(0.7, 12.0, s)
        assert ok[0] and abs(E[0] - Ec) < 1e-10 and abs(Lz[0] - Lc) < 1e-9 and abs(Q[0]) < 1e-12
