"""Pins of the oracle's convergence diagnostics (paper section 3, Fig. 4-9) against the paper's Table 1,
the closed-form epicyclic frequency, and the trajectory-based measurements of test_oracle_table1.  CPU only."""
import numpy as np
import pytest

import closed_forms as cf
import oracle
from conftest import load_table1
from test_oracle_table1 import delta_phi_first_cycle, first_peak_abs_costheta

ROWS = load_table1()
INF = float("inf")


def table1_state():
    xu8 = np.array([cf.spherical_photon_state(1.0, r["r"])[0] for r in ROWS])
    st = oracle.init_explicit(1.0, xu8, oracle.NULL)      # Table 1 are photon orbits given explicitly
    return st, xu8


def test_diagnostics_reproduce_table1_columns():
    st, _ = table1_state()
    stats, d = oracle.integrate_diagnostics(st, 24.0, oracle.step_control(mode=0, h_fixed=1.0 / 256, max_steps=10 ** 7))
    assert stats["n_active"] == 6 and stats["steps"] == 6 * 24 * 256
    for k, row in enumerate(ROWS):
        assert abs(d["cos_peak"][k] - row["maxcos"]) < 6e-5                      # PAPER.md:176-181, column 6
        dphi = d["dphi_cycle"][k]
        if row["label"] == "C":                                                  # crosses the pole: mod 2 pi
            dphi = (dphi - row["dphi"] + np.pi) % (2 * np.pi) - np.pi + row["dphi"]
        assert abs(dphi - row["dphi"]) < 6e-5                                    # column 7
    assert (d["max_abs_u2"] < 1e-7).all() and (d["max_abs_u2"] > 0).all()


def test_diagnostics_equal_the_trajectory_based_measurements():
    st, xu8 = table1_state()
    n = 64
    _, d = oracle.integrate_diagnostics(st, 20.0, oracle.step_control(mode=0, h_fixed=1.0 / n, max_steps=10 ** 7))
    for k in range(6):
        traj = oracle.trajectory(1.0, xu8[k], 1.0 / n, 20 * n)
        assert abs(d["cos_peak"][k] - first_peak_abs_costheta(traj, 1.0)) < 1e-13
        assert abs(d["dphi_cycle"][k] - delta_phi_first_cycle(traj, 1.0)) < 1e-11
        u2 = max(abs(oracle.invariants_one(1.0, 0, y)[3]) for y in traj)
        assert abs(d["max_abs_u2"][k] - u2) <= 1e-18 + 1e-12 * u2


def test_max_u2_converges_at_fourth_order():
    # PAPER.md:231, Fig. 5 (window inside the pre-blow-up regime, DESIGN R13)
    errs = []
    for n in (16, 32, 64, 128):
        st, _ = table1_state()
        _, d = oracle.integrate_diagnostics(st, 6.0, oracle.step_control(mode=0, h_fixed=1.0 / n, max_steps=10 ** 7))
        errs.append(d["max_abs_u2"])
    errs = np.array(errs)
    ratios = errs[:-1] / errs[1:]
    assert ((ratios > 8.0) & (ratios < 30.0)).all(), ratios


@pytest.mark.parametrize("a", [1.0, 0.9, 0.0])
def test_vertical_epicyclic_frequency_from_z_maxima(a):
    # PAPER.md:263-269, Fig. 9: v_z = 1e-12 kick, time between successive maxima of z(t)
    radii = np.array([4.0, 6.0, 9.0]) if a < 1 else np.array([1.4, 4.0, 9.0])
    if a == 0.0:
        radii = np.array([7.0, 9.0, 12.0])
    xu8 = np.array([cf.circular_orbit_state(a, r, +1, vz=1e-12) for r in radii])
    st = oracle.init_timelike(a, xu8)
    expect = np.array([cf.vertical_epicyclic(a, r, +1) for r in radii])
    ut = np.array([cf.circular_orbit(a, r, +1)[3] for r in radii])
    h = float(np.min(2 * np.pi / expect / ut) / 2048.0)
    nsteps = int(np.max(2 * np.pi / expect / ut) / h * 2.4)
    _, d = oracle.integrate_diagnostics(st, INF, oracle.step_control(mode=0, h_fixed=h, max_steps=nsteps))
    measured = 2 * np.pi / (d["t_zmax2"] - d["t_zmax1"])
    assert np.all(np.isfinite(measured)) and np.abs(measured / expect - 1.0).max() < 1e-6
    assert np.isnan(d["cos_peak"]).sum() == 0 and (d["cos_peak"] < 1e-10).all()   # tiny oscillation about the equator


def test_events_that_never_happen_are_nan():
    st = oracle.init_null(0.5, 50.0, np.radians(90.0), 5.0, 1e-9, 4, 1)     # equatorial rays: z stays ~0
    stats, d = oracle.integrate_diagnostics(st, INF, oracle.step_control(mode=1, eta=0.02, r_escape=60.0))
    assert stats["n_active"] == 0
    assert np.isnan(d["t_zmax2"]).all() and np.isfinite(d["max_abs_u2"]).all()
    # same final state as the plain driver loop
    ref = oracle.init_null(0.5, 50.0, np.radians(90.0), 5.0, 1e-9, 4, 1)
    oracle.integrate(ref, INF, oracle.step_control(mode=1, eta=0.02, r_escape=60.0))
    assert np.array_equal(ref.q, st.q) and np.array_equal(ref.nsteps, st.nsteps) and np.array_equal(ref.status, st.status)


def test_upward_zero_between_the_first_two_samples_counts():
    """gray2.h: dphi_cycle is taken at the first pair z_k < 0 <= z_{k+1}, k = 0, 1, ...  Start Table 1 row A
    half a step below the equator, moving up: the zero lies between samples 0 and 1.  The expected value is
    measured on the stored trajectory with numpy (nothing of the accumulator is reused)."""
    y0, _, _ = cf.spherical_photon_state(1.0, ROWS[0]["r"])
    h = 1.0 / 64
    back = oracle.trajectory(1.0, y0, -h, 1)[-1]                   # one step back: z < 0, u^z > 0
    start = 0.5 * (back + y0)
    start[4:] = y0[4:]
    assert start[3] < 0.0 < start[7]
    st = oracle.init_explicit(1.0, start[None, :], oracle.NULL)
    _, d = oracle.integrate_diagnostics(st, 2.0, oracle.step_control(mode=0, h_fixed=h, max_steps=10 ** 6))
    traj = oracle.trajectory(1.0, start, h, 128)
    z = traj[:, 3]
    assert z[0] < 0.0 <= z[1]
    r = np.array([oracle.ks_r(1.0, *p) for p in traj[:, 1:4]])
    phi = np.unwrap(np.arctan2(traj[:, 2], traj[:, 1]) - np.arctan2(1.0, r))
    w = -z[0] / (z[1] - z[0])
    expect = w * (phi[1] - phi[0])
    assert abs(d["dphi_cycle"][0] - expect) < 1e-13 and 0.0 < expect < 0.05
