"""Pins of the whole oracle integrator against the paper's worked example: Table 1 and the
convergence claims of section 3.1.  CPU only."""
import numpy as np
import pytest

import closed_forms as cf
import oracle
from conftest import load_table1

A_SPIN = 1.0  # Table 1 uses the extreme Kerr hole
ROWS = load_table1()


def ks_r_of(traj, a):
    return np.array([oracle.ks_r(a, *p) for p in traj[:, 1:4]])


def first_peak_abs_costheta(traj, a):
    """quadratic through the largest three samples around the first maximum."""
    c = np.abs(traj[:, 3] / ks_r_of(traj, a))
    i = 1
    while not (c[i] >= c[i - 1] and c[i] > c[i + 1]):
        i += 1
    y0, y1, y2 = c[i - 1], c[i], c[i + 1]
    return y1 - (y2 - y0) ** 2 / (8.0 * (y0 - 2.0 * y1 + y2))


def delta_phi_first_cycle(traj, a):
    """linear interpolation of the root of z(phi) at the first complete cycle.
    phi is the spherical KS angle: x + i y = (r + i a) sin(theta) e^{i phi}."""
    x, y, z = traj[:, 1], traj[:, 2], traj[:, 3]
    r = ks_r_of(traj, a)
    phi = np.unwrap(np.arctan2(y, x) - np.arctan2(a, r))
    k = next(j for j in range(1, len(z) - 1) if z[j] < 0.0 <= z[j + 1])
    w = -z[k] / (z[k + 1] - z[k])
    return phi[k] + w * (phi[k + 1] - phi[k]) - phi[0]


@pytest.mark.parametrize("row", ROWS, ids=[r["label"] for r in ROWS])
def test_closed_forms_reproduce_table1_columns(row):
    # pins closed_forms.teo_phi_q / max_abs_costheta themselves to the paper's printed numbers
    phi, q = cf.teo_phi_q(A_SPIN, row["r"])
    assert abs(phi - row["phi"]) < 5e-5
    assert abs(q - row["q"]) < 5e-5
    assert abs(cf.max_abs_costheta(A_SPIN, phi, q) - row["maxcos"]) < 5e-5
    assert cf.r_photon_prograde(A_SPIN) <= row["r"] <= cf.r_photon_retrograde(A_SPIN)


@pytest.mark.parametrize("row", ROWS, ids=[r["label"] for r in ROWS])
def test_invariants_of_table1_initial_data(row):
    y0, phi, q = cf.spherical_photon_state(A_SPIN, row["r"])
    E, Lz, Q, norm = oracle.invariants_one(A_SPIN, oracle.NULL, y0)
    assert abs(E - 1.0) < 1e-13
    assert abs(Lz - row["phi"]) < 5e-5 and abs(Lz - phi) < 1e-12
    assert abs(Q - row["q"]) < 5e-5 and abs(Q - q) < 1e-11
    assert abs(norm) < 1e-13          # "u^2 is initially of order 1e-16"


@pytest.mark.parametrize("row", ROWS, ids=[r["label"] for r in ROWS])
def test_integrator_reproduces_table1_max_costheta_and_delta_phi(row):
    y0, _, _ = cf.spherical_photon_state(A_SPIN, row["r"])
    n = 256
    traj = oracle.trajectory(A_SPIN, y0, 1.0 / n, 24 * n)
    assert abs(first_peak_abs_costheta(traj, A_SPIN) - row["maxcos"]) < 6e-5
    dphi = delta_phi_first_cycle(traj, A_SPIN)
    if row["label"] == "C":  # passes through the pole: phi jumps by pi there; compare mod 2 pi
        dphi = (dphi - row["dphi"] + np.pi) % (2 * np.pi) - np.pi + row["dphi"]
    assert abs(dphi - row["dphi"]) < 6e-5
    # the orbit stays on its sphere for the first cycle (unstable: error grows exponentially)
    assert np.abs(ks_r_of(traj[: 8 * n], A_SPIN) - row["r"]).max() < 1e-6


def test_test_c_passes_through_the_pole():
    # "exactly passes the poles ... at x = y = 0 and z ~ +-2.41", no special handling
    row = ROWS[2]
    y0, _, _ = cf.spherical_photon_state(A_SPIN, row["r"])
    traj = oracle.trajectory(A_SPIN, y0, 1.0 / 1024, 8 * 1024)
    rho = np.hypot(traj[:, 1], traj[:, 2])
    k = np.argmin(rho)
    assert rho[k] < 3e-3 and abs(abs(traj[k, 3]) - 2.41) < 0.01
    inv = np.array([oracle.invariants_one(A_SPIN, 0, y) for y in traj[max(k - 3, 0): k + 4]])
    assert np.all(np.isfinite(inv)) and np.abs(inv[:, 2] - row["q"]).max() < 1e-3


@pytest.mark.parametrize("label", ["A", "B", "E"])
def test_fourth_order_convergence_of_u2(label):
    # PAPER.md:231, Fig. 5: max|u^2| converges at 4th order.  Window 0 <= lambda <= 6 keeps the unstable
    # orbit in the pre-blow-up regime at every step size used here (coarse steps
    # leave the sphere and blow up; the paper's 0 <= lambda <= 64 window includes that regime).
    row = next(r for r in ROWS if r["label"] == label)
    y0, _, _ = cf.spherical_photon_state(A_SPIN, row["r"])
    errs = []
    for n in (16, 32, 64, 128):
        traj = oracle.trajectory(A_SPIN, y0, 1.0 / n, 6 * n)
        errs.append(max(abs(oracle.invariants_one(A_SPIN, 0, y)[3]) for y in traj))
    ratios = [errs[i] / errs[i + 1] for i in range(len(errs) - 1)]
    assert all(9.0 < q < 28.0 for q in ratios), (errs, ratios)


@pytest.mark.parametrize("label", ["A", "B", "D"])
def test_fourth_order_convergence_of_peak_and_delta_phi_and_position(label):
    # PAPER.md:247-249, Fig. 7-8
    row = next(r for r in ROWS if r["label"] == label)
    y0, phi, q = cf.spherical_photon_state(A_SPIN, row["r"])
    exact_peak = cf.max_abs_costheta(A_SPIN, phi, q)
    ref = oracle.trajectory(A_SPIN, y0, 1.0 / 1024, 16 * 1024)
    ref_dphi = delta_phi_first_cycle(ref, A_SPIN)
    pe, de, xe = [], [], []
    for n in (16, 32, 64, 128):
        traj = oracle.trajectory(A_SPIN, y0, 1.0 / n, 16 * n)
        pe.append(abs(first_peak_abs_costheta(traj, A_SPIN) - exact_peak))
        de.append(abs(delta_phi_first_cycle(traj, A_SPIN) - ref_dphi))
        xe.append(np.abs(traj[4 * n, 1:4] - ref[4 * 1024, 1:4]).max())   # position at lambda = 4
    for errs in (pe, de, xe):
        ratios = [errs[i] / errs[i + 1] for i in range(len(errs) - 1)]
        assert all(8.0 < r_ < 32.0 for r_ in ratios), (errs, ratios)


def test_u2_grows_and_smaller_step_is_smaller():
    # u^2 "increases approximately linearly"; "a smaller step size leads to smaller u^2"
    y0, _, _ = cf.spherical_photon_state(A_SPIN, 1.8)
    out = []
    for n in (16, 64):
        traj = oracle.trajectory(A_SPIN, y0, 1.0 / n, 12 * n, stride=n)
        out.append([abs(oracle.invariants_one(A_SPIN, 0, y)[3]) for y in traj])
    coarse, fine = np.array(out[0]), np.array(out[1])
    assert np.all(fine[2:] < coarse[2:])
    assert coarse[-1] > 3.0 * coarse[2]
