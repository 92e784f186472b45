"""GPU parity: the CUDA path, called through the C-ABI binding, against the oracle on the same seeded
inputs, element by element.  Tolerances: gpu_helpers.py (from BASELINE.json's north_star)."""
import numpy as np
import pytest
import torch

import image_helpers as ih
import oracle
from gpu_helpers import (INF, invariant_term_scales, TOL_DRIFT_F64, TOL_STATE_F32, TOL_STATE_F64, assert_fp32_parity, drift,
                         gpu_invariants_np, image_sc, image_sc_kw, make_straddle_check, run_gpu_image, run_oracle_image, sc_pair,
                         state_rel_error, take, to_oracle_state, twin_sensitivity)
from paper_1706_07062_b200 import gray2, inputs

pytestmark = pytest.mark.gpu


# ---- a3: the right-hand side alone ----------------------------------------------------------------

@pytest.mark.parametrize("a", [0.0, 0.5, -0.9375, 0.99, 1.0])
def test_rhs_matches_oracle_christoffel_form(a):
    rng = np.random.default_rng(7)
    n = 4099   # several blocks and a ragged tail
    pos = rng.uniform(-12, 12, (3, n))
    rr = np.array([oracle.ks_r(a, *pos[:, k]) for k in range(n)])
    pos[:, rr < 1.05 * (1 + np.sqrt(1 - a * a))] *= 6.0
    pos[:, 0] = [0.0, 0.0, 2.4]      # the pole
    pos[:, 1] = [3.0, -1.0, 0.0]     # the equator
    u = rng.uniform(-1, 1, (4, n))
    u[0] = rng.uniform(1, 3, n)
    expect = np.array([oracle.ks_accel(a, pos[:, k], u[:, k]) for k in range(n)]).T
    got = gray2.rhs(gray2.F64, a, torch.tensor(pos, device="cuda"), torch.tensor(u, device="cuda")).cpu().numpy()
    scale = np.abs(expect).max(axis=0, keepdims=True) + 1e-300
    assert np.max(np.abs(got - expect) / scale) < 2e-12
    got32 = gray2.rhs(gray2.F32, a, torch.tensor(pos, device="cuda"), torch.tensor(u, device="cuda")).cpu().numpy()
    assert np.max(np.abs(got32 - expect) / scale) < 2e-4


# ---- a1, a2: initial conditions -------------------------------------------------------------------

@pytest.mark.parametrize("cfg", [inputs.CFG1_NULL, inputs.CFG3_NULL.scaled(97, 61)], ids=lambda c: c.name)
def test_init_null_matches_oracle(cfg):
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    assert (g.a_eff, g.kind, g.reversed) == (o.a_eff, o.kind, o.reversed)
    gq = g.q.cpu().numpy()
    assert np.max(np.abs(gq - o.q) / np.maximum(np.abs(o.q), 1.0)) < 1e-14
    assert (g.status.cpu().numpy() == 0).all() and (g.nsteps.cpu().numpy() == 0).all() and (g.lam.cpu().numpy() == 0).all()
    g32 = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=gray2.F32)
    assert g32.q.dtype == torch.float32
    assert np.max(np.abs(g32.q.double().cpu().numpy() - o.q) / np.maximum(np.abs(o.q), 1.0)) < 1e-7


def test_init_timelike_matches_oracle():
    xu8, _ = inputs.cfg4_ensemble(1000)
    for renorm in (False, True):
        x = xu8.copy()
        if renorm:
            x[:, 4] = 99.0
        g = gray2.init_timelike(0.7, x, renormalise_ut=renorm)
        o = oracle.init_timelike(0.7, x, renormalise_ut=renorm)
        assert np.max(np.abs(g.q.cpu().numpy() - o.q) / np.maximum(np.abs(o.q), 1.0)) < 1e-14
        assert (g.a_eff, g.kind, g.reversed) == (0.7, gray2.TIMELIKE, 0)
    gi = gpu_invariants_np(gray2.init_timelike(0.7, xu8))
    oi = oracle.invariants(oracle.init_timelike(0.7, xu8))
    for a_, b_ in zip(gi, oi):
        assert np.max(np.abs(a_ - b_) / np.maximum(np.abs(b_), 1.0)) < 1e-13


def test_init_explicit_of_either_kind_matches_oracle(table1):
    """The paper's Table 1 orbits are explicit PHOTON data: through gray2_init_explicit with
    kind = NULL the state-level invariants are (1, Phi, Q, 0) with no patching of the struct; the kind decides
    mu^2 in Carter's Q and in the u^t solve, exactly as in the oracle."""
    import closed_forms as cf
    xu8 = np.array([cf.spherical_photon_state(1.0, r["r"])[0] for r in table1])
    moved = np.array([oracle.trajectory(1.0, y, 1.0 / 64, 40)[-1] for y in xu8])     # off the equator: mu^2 enters Q
    for kind in (gray2.NULL, gray2.TIMELIKE):
        for data in (xu8, moved):
            for renorm in (False, True):
                x = data.copy()
                if renorm:
                    x = x[[0, 2, 3, 4, 5]]            # rows B's start (r = 2, a = 1) is on the ergosphere: 1 - f = 0
                    x[:, 4] = 99.0
                g = gray2.init_explicit(1.0, x, kind, renormalise_ut=renorm)
                o = oracle.init_explicit(1.0, x, kind, renormalise_ut=renorm)
                assert (g.kind, g.reversed, g.a_eff) == (kind, 0, 1.0) == (o.kind, o.reversed, o.a_eff)
                assert np.max(np.abs(g.q.cpu().numpy() - o.q) / np.maximum(np.abs(o.q), 1.0)) < 1e-13
                for a_, b_ in zip(gpu_invariants_np(g), oracle.invariants(o)):
                    assert np.max(np.abs(a_ - b_) / np.maximum(np.abs(b_), 1.0)) < 1e-12
    E, Lz, Q, norm = gpu_invariants_np(gray2.init_explicit(1.0, xu8, gray2.NULL))
    for k, row in enumerate(table1):
        assert abs(E[k] - 1) < 1e-13 and abs(Lz[k] - row["phi"]) < 5e-5 and abs(Q[k] - row["q"]) < 5e-5 and abs(norm[k]) < 1e-13
    with pytest.raises(gray2.Gray2Error):
        gray2.init_explicit(1.0, xu8, 7)
    t = gray2.init_timelike(1.0, xu8)
    assert t.kind == gray2.TIMELIKE and torch.equal(t.q, gray2.init_explicit(1.0, xu8, gray2.TIMELIKE).q)


# ---- whole path on image configs ------------------------------------------------------------------

def compare_image(cfg, g0, g, o0, o, idx=None):
    """Shared checks for an image config; idx = the pixel indices the oracle ran (None = all)."""
    gst = to_oracle_state(g)
    if idx is not None:
        gst = take(gst, idx)
    full0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    d, mask = ih.classify_image(cfg, full0 if idx is None else full0)
    if idx is not None:
        d, mask = d[idx], mask[idx]
    outside = d > 1e-3
    # capture/escape flag and step count: bit-exact outside the band, vs the oracle AND vs Carter's potential
    assert np.array_equal(gst.status[outside], o.status[outside])
    assert np.array_equal(gst.nsteps[outside], o.nsteps[outside])
    assert np.array_equal((gst.status == gray2.CAPTURED)[outside], mask[outside])
    same = outside & (gst.nsteps == o.nsteps) & (gst.status == o.status)
    err = state_rel_error(gst.q[:, same], o.q[:, same], o.a_eff)
    assert err.max() < TOL_STATE_F64, err.max()
    assert np.max(np.abs(gst.lam[same] - o.lam[same]) / np.maximum(o.lam[same], 1.0)) < TOL_STATE_F64   # lambda = sum of eta r
    # invariant drift identical within 1e-12
    gi1 = gpu_invariants_np(g)
    gi0 = gpu_invariants_np(g0)
    if idx is not None:
        gi1 = [v[idx] for v in gi1]
        gi0 = [v[idx] for v in gi0]
    oi1, oi0 = oracle.invariants(o), oracle.invariants(o0)
    # a drift is a difference of two evaluations: the rounding of either end bounds what can agree
    scales = [np.maximum(s1, s0) for s1, s0 in zip(invariant_term_scales(o.q), invariant_term_scales(o0.q))]
    for k, (gd, od) in enumerate(zip(drift(gi1, gi0), drift(oi1, oi0))):
        scale = scales[k]
        # beside the term-scaled figure, the plain one: the difference of the two drifts relative to the drift itself
        # (rms over the rays) and the largest difference relative to max(1, |invariant|)
        rms_d = np.sqrt(np.mean(od[same] ** 2))
        print("[drift %s] %-3s rms drift %.2e; GPU - oracle: rms %.2e (%.1e of the drift), max %.2e of max(1,|value|), max %.2e of the terms"
              % (cfg.name, ("E", "Lz", "Q", "u.u")[k], rms_d, np.sqrt(np.mean((gd - od)[same] ** 2)),
                 np.sqrt(np.mean((gd - od)[same] ** 2)) / max(rms_d, 1e-300),
                 np.max(np.abs(gd - od)[same] / np.maximum(1.0, np.abs(oi0[k][same]))), np.max(np.abs(gd - od)[same] / scale[same])))
        assert np.max(np.abs(gd - od)[same] / scale[same]) < TOL_DRIFT_F64, (k, np.max(np.abs(gd - od)[same] / scale[same]))
    return outside, same


def test_cfg1_schwarzschild_image_full_parity():
    cfg = inputs.CFG1_NULL
    g0, g, gstats = run_gpu_image(cfg)
    o0, o, ostats = run_oracle_image(cfg)
    outside, same = compare_image(cfg, g0, g, o0, o)
    assert outside.mean() > 0.995 and same.sum() == outside.sum()
    assert gstats["n_active"] == 0 and gstats["n_invalid"] == 0 and gstats["n_maxsteps"] == 0
    assert gstats["steps"] == int(g.nsteps.sum().item())
    if outside.all():
        assert gstats == ostats


def test_cfg1_timelike_orbits_parity():
    xu8, r0 = inputs.cfg1_orbits()
    gsc, osc = sc_pair(mode=0, h_fixed=0.5, max_steps=5000)
    g = gray2.init_timelike(0.0, xu8)
    g0 = g.clone()
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    o = oracle.init_timelike(0.0, xu8)
    o0 = o.copy()
    oracle.integrate(o, INF, osc)
    gst = to_oracle_state(g)
    assert (gst.status == gray2.MAXSTEPS).all() and (gst.nsteps == 5000).all()
    assert gray2.stats_dict(stats) == dict(steps=80000, n_captured=0, n_escaped=0, n_maxsteps=16, n_invalid=0, n_active=0)
    assert state_rel_error(gst.q, o.q, 0.0).max() < TOL_STATE_F64
    assert np.max(np.abs(gst.lam - 2500.0)) < 1e-9
    gd = drift(gpu_invariants_np(g), gpu_invariants_np(g0))
    od = drift(oracle.invariants(o), oracle.invariants(o0))
    for a_, b_ in zip(gd, od):
        assert np.max(np.abs(a_ - b_)) < 1e-11   # 5000 steps of fixed h: both drifts ~1e-9, equal to 1e-11


@pytest.mark.parametrize("cfg", [inputs.CFG2_NULL.scaled(96, 80), inputs.CFG3_NULL.scaled(131, 77),
                                 inputs.CFG5_NULL.scaled(100, 100)], ids=lambda c: c.name)
def test_kerr_images_reduced_resolution_full_parity(cfg):
    g0, g, gstats = run_gpu_image(cfg)
    o0, o, ostats = run_oracle_image(cfg)
    outside, same = compare_image(cfg, g0, g, o0, o)
    assert outside.mean() > 0.99
    assert gstats["n_active"] == 0 and gstats["n_invalid"] == 0
    assert abs(gstats["steps"] - ostats["steps"]) <= 40 * (~outside).sum()


@pytest.mark.parametrize("launch", [(0, 0), (256, 2)], ids=["default-launch", "packed-256x2"])
@pytest.mark.parametrize("cfg", [inputs.CFG3_NULL.scaled(64), inputs.CFG1_NULL, inputs.CFG2_NULL.scaled(72, 56)],
                         ids=lambda c: c.name)
def test_fp32_against_oracle(cfg, launch):
    """north_star's FP32 clause on EVERY non-critical ray, all eight components (DESIGN R12; gpu_helpers).  Images this
    small get the one-per-thread float kernel by default (gray2_abi.cu, small batches); the second launch forces the
    packed two-per-thread kernel that full-size images -- and bench.py -- run.  (The coordinate-time and
    Boyer-Lindquist forms have the packed kernel only, at every size.)"""
    gray2.set_launch(gray2.F32, *launch)
    try:
        g0, g, gstats = run_gpu_image(cfg, prec=gray2.F32)
    finally:
        gray2.set_launch(gray2.F32, 0, 0)
    o0 = to_oracle_state(g0)                        # the same inputs: the float initial state, widened
    o = o0.copy()
    kw = image_sc_kw(cfg)
    oracle.integrate(o, INF, oracle.step_control(**kw))
    gst = to_oracle_state(g)
    sens = twin_sensitivity(o0, kw)
    err = state_rel_error(gst.q, o.q, o.a_eff)
    noncrit, same = assert_fp32_parity(cfg.name, gst, o, sens, err, make_straddle_check(o0, gst, o, kw))
    # the capture mask against Carter's potential, from the constants of the rounded input
    xi, eta, _, _ = ih.ray_constants(o0)
    mask = ih.potential_mask(o0.a_eff, xi, eta, 0.9 * cfg.r_obs)
    assert np.array_equal((gst.status == gray2.CAPTURED)[noncrit], mask[noncrit])
    assert gstats["n_active"] == 0 and gstats["n_invalid"] == 0


def degenerate_band_distance(cfg, o0):
    """Distance of every ray to the critical curve in the asymptotic image plane for the cases the general band
    machinery does not cover (it needs sin i != 0 and |a| < 1), from closed forms and the ray constants
    (xi, eta) of the oracle's initial state:
      face-on (sin i = 0): every ray has xi = 0 and the picture is axisymmetric, so the curve is the circle of
        radius sqrt(eta_c + a^2), eta_c = Q(r_0) at the spherical photon orbit with Phi(r_0) = 0 (a = 0: sqrt 27),
        and a ray sits at radius sqrt(eta + a^2);
      extremal spin: Phi(r) = -(r^2 - 2r - 1), Q(r) = -r^3 (r - 4) for 1 < r <= 4, plus the vertical segment
        alpha = -2 / sin i, |beta| <= sqrt(3 + cos^2 i - 4 cot^2 i), onto which all of r -> 1 is mapped."""
    import closed_forms as cf
    xi, eta, _, _ = ih.ray_constants(o0)
    a, inc = abs(cfg.a), cfg.inclination
    if abs(np.sin(inc)) < 1e-12:
        assert np.abs(xi).max() < 1e-9
        if a == 0.0:
            rc = np.sqrt(27.0)
        else:
            lo, hi = cf.r_photon_prograde(a), cf.r_photon_retrograde(a)
            for _ in range(200):                        # bisection on Phi(r) = 0
                mid = 0.5 * (lo + hi)
                lo, hi = (mid, hi) if cf.teo_phi_q(a, mid)[0] > 0 else (lo, mid)
            rc = np.sqrt(cf.teo_phi_q(a, lo)[1] + a * a)
        return np.abs(np.sqrt(np.maximum(eta + a * a, 0.0)) - rc)
    assert a == 1.0
    r = np.linspace(1.0, 4.0, 400001)[1:]
    cxi, ceta = -(r * r - 2 * r - 1), -r ** 3 * (r - 4)
    b2 = ceta + np.cos(inc) ** 2 - cxi ** 2 / np.tan(inc) ** 2
    ca, cb = -cxi[b2 >= 0] / np.sin(inc), np.sqrt(b2[b2 >= 0])
    seg = np.sqrt(max(3.0 + np.cos(inc) ** 2 - 4.0 / np.tan(inc) ** 2, 0.0))
    ca = np.concatenate([ca, np.full(20001, -2.0 / np.sin(inc))])
    cb = np.concatenate([cb, np.linspace(0.0, seg, 20001)])
    _, beta = ih.pixel_grid(cfg)
    al, be = ih.asymptotic_image_point(o0.a_eff, inc, xi, eta, np.where(beta >= 0, 1.0, -1.0))
    if cfg.a < 0:
        ca = -ca
    d = np.empty(al.size)
    for lo in range(0, al.size, 256):
        hi = min(lo + 256, al.size)
        d[lo:hi] = np.sqrt(np.min((ca[None, :] - al[lo:hi, None]) ** 2 + (cb[None, :] - np.abs(be[lo:hi, None])) ** 2, axis=1))
    return d


@pytest.mark.parametrize("a,inc_deg", [(1.0, 80.0), (0.9375, 0.0), (-0.99, 180.0), (0.0, 0.0)],
                         ids=["extremal-spin", "face-on", "face-on-from-below-retrograde", "schwarzschild-pole"])
def test_degenerate_geometries(a, inc_deg):
    """Extremal spin, and the face-on view in which the rays run along the spin axis through the poles
    (the case that crashes Boyer-Lindquist integrators): no special handling exists or is
    needed.  Status and step count must equal the oracle's on EVERY ray further than 1e-3 M from the critical
    curve (closed forms for these four cases: degenerate_band_distance), the states to 1e-9."""
    cfg = inputs.NullImageConfig("t", a, 1000.0, inc_deg, 9.0, 64, 48)
    g0, g, gstats = run_gpu_image(cfg)
    o0, o, ostats = run_oracle_image(cfg)
    gst = to_oracle_state(g)
    d = degenerate_band_distance(cfg, o0)
    outside = d > 1e-3
    assert outside.mean() > 0.99, outside.mean()
    assert np.array_equal(gst.status[outside], o.status[outside])
    assert np.array_equal(gst.nsteps[outside], o.nsteps[outside])
    differ = (gst.nsteps != o.nsteps) | (gst.status != o.status)
    print("[degenerate %s] %d rays inside the band, %d of them differ from the oracle" % (cfg.name, (~outside).sum(), differ.sum()))
    same = ~differ
    assert state_rel_error(gst.q[:, same], o.q[:, same], o.a_eff).max() < TOL_STATE_F64
    assert gstats["n_invalid"] == 0 and gstats["n_active"] == 0 and gstats["n_maxsteps"] == ostats["n_maxsteps"]
    if inc_deg in (0.0, 180.0):
        # axisymmetry about the line of sight: the captured region is a disc centred on the image centre
        alpha, beta = ih.pixel_grid(cfg)
        b = np.hypot(alpha, beta)
        cap = gst.status == gray2.CAPTURED
        assert b[cap].max() < b[~cap].min() + 2 * cfg.fov / 48
