"""Pins of the oracle's image-plane initial conditions and of the whole null-ray pipeline:
Bardeen's shadow boundary and Carter's radial potential (closed_forms F6, F7).  CPU only."""
import numpy as np
import pytest

import closed_forms as cf
import image_helpers as ih
import oracle
from paper_1706_07062_b200 import inputs

INF = float("inf")


def run_image(cfg):
    st0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    st = st0.copy()
    sc = oracle.step_control(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                             capture_factor=cfg.capture_factor)
    stats = oracle.integrate(st, INF, sc)
    return st0, st, stats


def test_init_null_geometry_and_index_order():
    a, r_obs, inc, W, nx, ny = 0.6, 200.0, np.radians(35.0), 9.0, 6, 4
    st = oracle.init_null(a, r_obs, inc, W, 2 * W, nx, ny)
    assert st.a_eff == -a and st.reversed == 1 and st.kind == oracle.NULL
    assert (st.status == oracle.ACTIVE).all() and (st.nsteps == 0).all() and (st.lam == 0).all()
    n = np.array([np.sin(inc), 0.0, np.cos(inc)])
    pos = st.q[1:4].T
    vel = st.q[5:8].T
    assert np.allclose(vel, -n[None, :], atol=1e-15)             # parallel rays, unit Euclidean tangent
    assert np.allclose(pos @ n, r_obs, atol=1e-12)               # all pixels in the plane at distance r_obs
    alpha = pos[:, 1]                                            # e_alpha = +y
    beta = (pos - r_obs * n[None, :]) @ np.array([-np.cos(inc), 0.0, np.sin(inc)])
    ea = -W + (np.arange(nx) + 0.5) * 2 * W / nx
    eb = -2 * W + (np.arange(ny) + 0.5) * 4 * W / ny
    assert np.allclose(alpha.reshape(ny, nx), ea[None, :].repeat(ny, 0), atol=1e-12)   # j fastest
    assert np.allclose(beta.reshape(ny, nx), eb[:, None].repeat(nx, 1), atol=1e-12)
    assert (st.q[0] == 0).all() and (st.q[4] > 0).all()


@pytest.mark.parametrize("a,inc_deg", [(0.9375, 60.0), (0.5, 30.0), (-0.8, 75.0)])
def test_init_null_conserved_quantities(a, inc_deg):
    # null, E = 1 + O(1/r_obs), and xi = Lz/E = -alpha sin(i) for the PHYSICAL photon (run value: +alpha sin i)
    inc = np.radians(inc_deg)
    r_obs = 1000.0
    cfg = inputs.NullImageConfig("t", a, r_obs, inc_deg, 12.0, 16, 16)
    st = oracle.init_null(a, r_obs, inc, 12.0, 12.0, 16, 16)
    E, Lz, Q, norm = oracle.invariants(st)
    alpha, beta = ih.pixel_grid(cfg)
    assert np.abs(norm).max() < 1e-13
    assert np.abs(E - 1.0).max() < 3.0 / r_obs
    assert np.abs(Lz - alpha * np.sin(inc)).max() < 1e-5   # Lz = x u_y - y u_x, u_i = u^i + f l_i U, f ~ 2/r_obs
    # (alpha, beta) are Bardeen's impact parameters up to O(1/r_obs)
    a_inf, b_inf = ih.asymptotic_image_point(st.a_eff, inc, Lz / E, Q / E ** 2, np.sign(beta))
    assert np.abs(a_inf - alpha).max() < 0.05 and np.abs(b_inf - beta).max() < 0.05


@pytest.mark.parametrize("inc_deg", [10.0, 60.0, 90.0])
def test_schwarzschild_shadow_is_a_disc_of_radius_sqrt27(inc_deg):
    cfg = inputs.NullImageConfig("t", 0.0, 1000.0, inc_deg, 7.0, 40, 40, r_escape=1100.0)
    st0, st, stats = run_image(cfg)
    alpha, beta = ih.pixel_grid(cfg)
    b = np.hypot(alpha, beta)
    cap = st.status == oracle.CAPTURED
    assert stats["n_captured"] + stats["n_escaped"] == cfg.n
    bc = np.sqrt(27.0)
    assert cap[b < bc - 0.02].all() and (~cap[b > bc + 0.02]).all()
    # exact conserved impact parameter b = sqrt(xi^2 + eta) decides, with no band at all at this resolution
    xi, eta, _, _ = ih.ray_constants(st0)
    assert np.array_equal(cap, np.sqrt(xi ** 2 + eta) < bc)


def test_mask_is_mirror_symmetric_in_beta():
    cfg = inputs.NullImageConfig("t", 0.9, 500.0, 50.0, 8.0, 24, 24, r_escape=600.0)
    _, st, _ = run_image(cfg)
    img = st.status.reshape(cfg.ny, cfg.nx)
    assert np.array_equal(img, img[::-1, :])
    # (the two rays share (xi, eta), hence R(r) and the capture flag, but not theta(lambda), so step counts differ)


def test_bardeen_closed_form_edges():
    # a = 0: circle of radius sqrt(27); a = 0.9375, i = 60 deg: values quoted in SURVEY.md 8(c) F6
    lo, hi = cf.bardeen_edges_on_axis(0.9375, np.radians(60.0))
    assert abs(lo + 2.92087) < 2e-5 and abs(hi - 6.64228) < 2e-5
    # extreme Kerr seen edge-on: prograde edge at alpha = -2 (r_p = 1 -> xi = 2), retrograde at +7 (r_r = 4 -> xi = -7)
    phi_p, _ = cf.teo_phi_q(1.0, cf.r_photon_retrograde(1.0))
    assert abs(phi_p + 7.0) < 1e-12


@pytest.mark.parametrize("a,inc_deg", [(0.9375, 60.0), (-0.9375, 60.0), (0.5, 30.0)])
def test_shadow_edges_on_the_alpha_axis_match_bardeen(a, inc_deg):
    """One image row through beta ~ 0: the captured interval must be Bardeen's, to a pixel and O(1/r_obs)."""
    inc = np.radians(inc_deg)
    nx = 2048
    cfg = inputs.NullImageConfig("t", a, 1000.0, inc_deg, 8.0, nx, 1)
    st0 = oracle.init_null(a, cfg.r_obs, inc, cfg.fov, 1e-9, nx, 1)
    st = st0.copy()
    oracle.integrate(st, INF, oracle.step_control(mode=1, eta=0.01, r_escape=1100.0, max_steps=20000))
    alpha = -cfg.fov + (np.arange(nx) + 0.5) * 2 * cfg.fov / nx
    cap = st.status == oracle.CAPTURED
    lo, hi = cf.bardeen_edges_on_axis(abs(a), inc)
    if a < 0:
        lo, hi = -hi, -lo
    tol = 2 * cfg.fov / nx + 0.02          # one pixel + finite-distance correction of the pixel <-> xi map
    assert abs(alpha[cap].min() - lo) < tol and abs(alpha[cap].max() - hi) < tol
    assert cap[(alpha > lo + tol) & (alpha < hi - tol)].all()
    # sharper, using the conserved xi of each ray instead of its pixel coordinate (no 1/r_obs error):
    xi, eta, _, _ = ih.ray_constants(st0)
    a_inf = xi / np.sin(inc)
    assert abs(a_inf[cap].min() - lo) < 2 * cfg.fov / nx and abs(a_inf[cap].max() - hi) < 2 * cfg.fov / nx


@pytest.mark.parametrize("cfg", [inputs.CFG1_NULL, inputs.CFG2_NULL.scaled(48), inputs.CFG3_NULL.scaled(48),
                                 inputs.CFG5_NULL.scaled(48)], ids=lambda c: c.name)
def test_capture_mask_equals_carter_potential_outside_the_band(cfg):
    """DESIGN R11 / north_star: outside 1e-3 M of the critical curve the mask is unique; it must equal the
    ODE-free classifier F7 for every such ray."""
    st0, st, stats = run_image(cfg)
    assert stats["n_maxsteps"] == 0 and stats["n_invalid"] == 0 and stats["n_active"] == 0
    d, mask = ih.classify_image(cfg, st0)
    outside = d > 1e-3
    assert outside.mean() > 0.99
    cap = st.status == oracle.CAPTURED
    assert np.array_equal(cap[outside], mask[outside])
    frac = cap.mean()
    assert 0.02 < frac < 0.35
    # invariants are conserved to RK4 truncation along every ray that is not within the band
    E0, L0, Q0, n0 = oracle.invariants(st0)
    E1, L1, Q1, n1 = oracle.invariants(st)
    esc = (st.status == oracle.ESCAPED) & outside
    assert np.abs(E1 - E0)[esc].max() < 1e-6 and np.abs(L1 - L0)[esc].max() < 1e-5
    assert np.abs(Q1 - Q0)[esc].max() < 1e-4 and np.abs(n1)[esc].max() < 1e-6
