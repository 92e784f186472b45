"""GPU parity of the Boyer-Lindquist variant (eq. 1, Table 2 "BL" rows): the
right-hand side, the KS <-> BL map, the invariants and the whole integration, through the C-ABI binding,
against the oracle's BL path (generic connection of eq. 1) on the same seeded inputs, element by element.
Tolerances: gpu_helpers.py.  On BL states the capture test also covers the RK4 stage positions (DESIGN R20);
rays whose polar turning point comes closer to the axis than sin(theta) = 0.05 are outside the domain in which
h = eta r resolves the BL equations (DESIGN R21) and are left out of the comparisons."""
import numpy as np
import pytest
import torch

import image_helpers as ih
import oracle
from gpu_helpers import (INF, TOL_STATE_F32, TOL_STATE_F64, assert_fp32_parity, drift, gpu_invariants_np, sc_pair,
                         state_rel_error, state_rel_error_bl, take, to_oracle_state, twin_sensitivity)
from paper_1706_07062_b200 import gray2, inputs

pytestmark = pytest.mark.gpu

BL_CAPTURE = 1.01
AXIS_MARGIN = 0.05
# Captured rays are stored next to the horizon, where u^t and u^phi grow like 1/Delta and Delta = P - 2r is a
# difference of nearly equal numbers (Delta ~ 0.003 ... 0.02 from terms ~2.5): a rounding-level difference in r
# shows up several hundred times larger in those components.  Escaped rays keep the 1e-9 of north_star.
TOL_STATE_BL_CAPTURED = 1e-7


def bl_sc_kw(cfg, **kw):
    args = dict(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps, capture_factor=BL_CAPTURE)
    args.update(kw)
    return args


def bl_sc(cfg, **kw):
    return sc_pair(**bl_sc_kw(cfg, **kw))


def bl_straddle_check(o0, gst, o, kw, rel=2e-5):
    """straddles(k) for Boyer-Lindquist states: at the smaller of the two step counts the oracle's r is within FP32
    rounding of r_escape, or the guarded step (DESIGN R20) changes its verdict when the capture radius moves by
    `rel` -- some stage of that step lies within FP32 rounding of the capture radius."""
    r_cap = kw["capture_factor"] * (1.0 + np.sqrt(1.0 - o0.a_eff ** 2))

    def straddles(k):
        n = min(int(gst.nsteps[k]), int(o.nsteps[k]))
        one = take(o0, [k])
        run = dict(kw)
        run.update(max_steps=n, r_escape=INF, capture_factor=1e-9)
        oracle.integrate(one, INF, oracle.step_control(**run))
        y = one.q[:, 0].copy()
        if abs(y[1] / kw["r_escape"] - 1.0) < rel or abs(y[1] / r_cap - 1.0) < rel:
            return True
        h = kw["eta"] * y[1]
        return oracle.bl_rk4_step_guarded(o0.a_eff, y, h, r_cap * (1 - rel))[0] != \
            oracle.bl_rk4_step_guarded(o0.a_eff, y, h, r_cap * (1 + rel))[0]
    return straddles


def bl_fp32_tolerances(o):
    """Per-ray factor on the FP32 tolerance: captured rays are stored next to the horizon, where u^t and u^phi
    grow like 1/Delta (see TOL_STATE_BL_CAPTURED: the same factor 100 as in double)."""
    return np.where(o.status == oracle.CAPTURED, TOL_STATE_BL_CAPTURED / TOL_STATE_F64, 1.0)


# ---- the right-hand side alone --------------------------------------------------------------------

@pytest.mark.parametrize("a", [0.0, 0.5, -0.9375, 0.99, 1.0])
def test_bl_rhs_matches_oracle_connection_of_eq1(a):
    rng = np.random.default_rng(11)
    n = 4099
    rp = 1.0 + np.sqrt(1.0 - a * a)
    r = 1.03 * rp + rng.uniform(0, 1, n) ** 3 * 60.0
    th = rng.uniform(0.02, np.pi - 0.02, n)
    th[:7] = [np.pi / 2, 0.02, np.pi - 0.02, -1.0, 4.0, 7.5, -5.3]      # equator, near the axis, outside [0, pi]
    u = rng.uniform(-1, 1, (4, n))
    u[0] = rng.uniform(1, 3, n)
    u[2:] /= r
    pos = np.stack([r, th])
    expect = np.array([oracle.bl_accel(a, [0.0, r[k], th[k], 0.0], u[:, k]) for k in range(n)]).T
    # angular accelerations carry a factor 1/r: weigh them by r, then compare with the largest component
    w = np.stack([np.ones(n), np.ones(n), r, r])
    scale = np.abs(expect * w).max(axis=0, keepdims=True) + 1e-300
    got = gray2.rhs_bl(gray2.F64, a, torch.tensor(pos, device="cuda"), torch.tensor(u, device="cuda")).cpu().numpy()
    assert np.max(np.abs(got - expect) * w / scale) < 5e-12
    got32 = gray2.rhs_bl(gray2.F32, a, torch.tensor(pos, device="cuda"), torch.tensor(u, device="cuda")).cpu().numpy()
    assert np.quantile(np.abs(got32 - expect) * w / scale, 0.999) < 2e-4


# ---- the coordinate map and the invariants ----------------------------------------------------------

@pytest.mark.parametrize("a,inc", [(0.9375, 60.0), (0.0, 60.0), (1.0, 80.0), (-0.5, 30.0)])
def test_convert_matches_oracle_both_ways(a, inc):
    cfg = inputs.NullImageConfig("t", a, 1000.0, inc, 12.0, 61, 47)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    gb, ob = gray2.convert(g, gray2.BL), oracle.convert(o, oracle.BL)
    assert (gb.coords, gb.a_eff, gb.kind, gb.reversed) == (gray2.BL, o.a_eff, o.kind, o.reversed)
    assert state_rel_error_bl(gb.q.cpu().numpy(), ob.q).max() < 1e-13
    for x, y in zip(gpu_invariants_np(gb), oracle.invariants(ob)):
        assert np.max(np.abs(x - y) / np.maximum(1.0, np.abs(y))) < 1e-10
    for x, y in zip(gpu_invariants_np(gb), gpu_invariants_np(g)):            # scalars: same in both systems
        assert np.max(np.abs(x - y) / np.maximum(1.0, np.abs(y))) < 1e-9
    gk = gray2.convert(gb, gray2.KS)
    ok = oracle.convert(ob, oracle.KS)
    assert gk.coords == gray2.KS
    assert state_rel_error(gk.q.cpu().numpy(), ok.q, o.a_eff).max() < 1e-13
    assert state_rel_error(gk.q.cpu().numpy(), o.q, o.a_eff).max() < 1e-12    # round trip
    assert torch.equal(gk.status, g.status) and torch.equal(gk.nsteps, g.nsteps) and torch.equal(gk.lam, g.lam)


def test_convert_near_the_hole_timelike_and_fp32():
    xu8, _ = inputs.cfg4_ensemble(3000)
    g = gray2.init_timelike(0.7, xu8)
    o = oracle.init_timelike(0.7, xu8)
    gb, ob = gray2.convert(g, gray2.BL), oracle.convert(o, oracle.BL)
    assert state_rel_error_bl(gb.q.cpu().numpy(), ob.q).max() < 1e-13
    for x, y in zip(gpu_invariants_np(gb), oracle.invariants(ob)):
        assert np.max(np.abs(x - y) / np.maximum(1.0, np.abs(y))) < 1e-12
    g32 = gray2.init_timelike(0.7, xu8, prec=gray2.F32)
    gb32 = gray2.convert(g32, gray2.BL)
    assert gb32.q.dtype == torch.float32 and gb32.coords == gray2.BL
    assert state_rel_error_bl(gb32.q.double().cpu().numpy(), ob.q).max() < 2e-6


def test_convert_in_place():
    cfg = inputs.CFG3_NULL.scaled(50, 40)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    ref = gray2.convert(g, gray2.BL)
    same = gray2.convert(g, gray2.BL, out=g)            # dst is src
    assert same is g and g.coords == gray2.BL and torch.equal(g.q, ref.q)
    back = gray2.convert(g, gray2.KS, out=g)
    assert back.coords == gray2.KS and torch.equal(back.q, gray2.convert(ref, gray2.KS).q)


def test_convert_and_coords_argument_checks():
    g = gray2.init_null(0.5, 1000.0, 1.0, 5.0, 5.0, 8, 8)
    with pytest.raises(gray2.Gray2Error) as e:
        gray2.convert(g, gray2.KS)
    assert e.value.code == gray2.EINVAL
    gb = gray2.convert(g, gray2.BL)
    with pytest.raises(gray2.Gray2Error):
        gray2.convert(gb, gray2.BL)
    with pytest.raises(gray2.Gray2Error):
        gray2.convert(g, gray2.BL, out=gray2.State.empty(64, gray2.F32))     # precision mismatch
    with pytest.raises(gray2.Gray2Error) as e:
        gray2.convert(g, gray2.BL, n=65)
    assert e.value.code == gray2.ESTATE
    sc = gray2.step_control(mode=1, eta=0.01, r_escape=1100.0, max_steps=5)
    with pytest.raises(gray2.Gray2Error) as e:
        gray2.integrate_coordtime(gb, 10.0, sc)
    assert e.value.code == gray2.EINVAL
    bad = gb.clone()
    bad.coords = 7
    with pytest.raises(gray2.Gray2Error):
        gray2.integrate(bad, INF, sc)


# ---- whole path on image configs --------------------------------------------------------------------

def run_pair(cfg, prec=gray2.F64, **kw):
    gsc, osc = bl_sc(cfg, **kw)
    g0 = gray2.convert(gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec), gray2.BL)
    g = g0.clone()
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    o0 = oracle.convert(oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny), oracle.BL)
    o = o0.copy()
    ostats = oracle.integrate(o, INF, osc)
    torch.cuda.synchronize()
    return g0, g, gray2.stats_dict(stats), o0, o, ostats


@pytest.mark.parametrize("cfg", [inputs.CFG1_NULL, inputs.CFG2_NULL.scaled(96, 80), inputs.CFG3_NULL.scaled(131, 77),
                                 inputs.CFG5_NULL.scaled(100, 100)], ids=lambda c: c.name)
def test_bl_images_full_parity(cfg):
    g0, g, gstats, o0, o, ostats = run_pair(cfg)
    gst = to_oracle_state(g)
    assert gst.coords == oracle.BL
    k0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    d, mask = ih.classify_image(cfg, k0)
    outside = (d > 1e-3) & (ih.axis_approach(k0) >= AXIS_MARGIN)
    assert outside.mean() > 0.9
    # capture/escape flag and step count: bit-exact outside the band, vs the oracle AND vs Carter's potential
    assert np.array_equal(gst.status[outside], o.status[outside])
    assert np.array_equal(gst.nsteps[outside], o.nsteps[outside])
    assert np.array_equal((gst.status == gray2.CAPTURED)[outside], mask[outside])
    assert gstats["n_active"] == 0
    assert gstats["steps"] == int(g.nsteps.sum().item())
    cap = outside & (gst.status == gray2.CAPTURED)      # stored at the last state outside the capture radius
    assert (gst.q[1][cap] >= BL_CAPTURE * (1.0 + np.sqrt(1.0 - cfg.a ** 2))).all()
    same = outside & (gst.nsteps == o.nsteps) & (gst.status == o.status)
    err = state_rel_error_bl(gst.q[:, same], o.q[:, same])
    captured = (o.status == oracle.CAPTURED)[same]
    assert err[~captured].max() < TOL_STATE_F64, (err[~captured].max(), np.quantile(err, [0.5, 0.99]))
    assert err[captured].max() < TOL_STATE_BL_CAPTURED and np.quantile(err[captured], 0.9) < TOL_STATE_F64
    assert np.max(np.abs(gst.lam[same] - o.lam[same]) / np.maximum(o.lam[same], 1.0)) < TOL_STATE_F64
    # invariant drift: the same on both sides to the rounding of the terms the invariants are sums of
    gd = drift(gpu_invariants_np(g), gpu_invariants_np(g0))
    od = drift(oracle.invariants(o), oracle.invariants(o0))
    r_end, r_start = o.q[1], o0.q[1]
    np.seterr(over="ignore", invalid="ignore")         # the rays lost near the axis hold overflowed values
    for k, (x, y) in enumerate(zip(gd, od)):
        # terms: E ~ u^t, L_z ~ r^2 u^phi, Q ~ (r^2 u^theta)^2 + L_z^2 cot^2, norm ~ (u^t)^2
        ut = np.maximum(np.abs(o.q[4]), np.abs(o0.q[4]))
        L = np.maximum(r_end ** 2 * np.hypot(o.q[6], o.q[7]), r_start ** 2 * np.hypot(o0.q[6], o0.q[7]))
        scale = [np.maximum(1.0, ut), np.maximum(1.0, L), np.maximum(1.0, L * L), np.maximum(1.0, ut * ut)][k]
        # (escaped rays: next to the horizon the invariants are differences of terms ~1/Delta)
        sel = same & (o.status == oracle.ESCAPED)
        assert np.max(np.abs(x - y)[sel] / scale[sel]) < 1e-11, (k, np.max(np.abs(x - y)[sel] / scale[sel]))


@pytest.mark.parametrize("cfg", [inputs.CFG3_NULL.scaled(64), inputs.CFG1_NULL], ids=lambda c: c.name)
def test_bl_fp32_against_oracle(cfg):
    """north_star's FP32 clause on every non-critical ray away from the axis (DESIGN R12, R21)."""
    kw = bl_sc_kw(cfg)
    ks32 = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=gray2.F32)
    g = gray2.convert(ks32, gray2.BL)
    o0 = to_oracle_state(g)                              # the same inputs: the float BL initial state, widened
    gray2.integrate(g, INF, gray2.step_control(**kw))
    o = o0.copy()
    oracle.integrate(o, INF, oracle.step_control(**kw))
    gst = to_oracle_state(g)
    k0 = to_oracle_state(ks32)
    sens = twin_sensitivity(k0, kw)                      # a property of the geodesic: measured in Kerr-Schild
    noncrit, same = assert_fp32_parity(cfg.name + " Boyer-Lindquist", gst, o, sens, state_rel_error_bl(gst.q, o.q),
                                       bl_straddle_check(o0, gst, o, kw), usable=ih.axis_approach(k0) >= AXIS_MARGIN,
                                       tol_scale=bl_fp32_tolerances(o))
    xi, eta, _, _ = ih.ray_constants(k0)
    mask = ih.potential_mask(k0.a_eff, xi, eta, 0.9 * cfg.r_obs)
    assert np.array_equal((gst.status == gray2.CAPTURED)[noncrit], mask[noncrit])


def test_bl_timelike_orbits_fixed_step_parity():
    xu8, r0 = inputs.cfg1_orbits()
    gsc, osc = sc_pair(mode=0, h_fixed=0.5, max_steps=3000, capture_factor=BL_CAPTURE)
    g0 = gray2.convert(gray2.init_timelike(0.0, xu8), gray2.BL)
    g = g0.clone()
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    o0 = oracle.convert(oracle.init_timelike(0.0, xu8), oracle.BL)
    o = o0.copy()
    oracle.integrate(o, INF, osc)
    gst = to_oracle_state(g)
    assert (gst.status == gray2.MAXSTEPS).all() and (gst.nsteps == 3000).all()
    assert gray2.stats_dict(stats) == dict(steps=48000, n_captured=0, n_escaped=0, n_maxsteps=16, n_invalid=0, n_active=0)
    assert state_rel_error_bl(gst.q, o.q).max() < TOL_STATE_F64
    assert np.max(np.abs(gst.q[1] - r0) / r0) < 1e-3          # circular orbits stay circular


def test_bl_kerr_ensemble_parity():
    xu8, _ = inputs.cfg4_ensemble(2000)
    gsc, osc = sc_pair(mode=0, h_fixed=0.5, max_steps=400, capture_factor=BL_CAPTURE)
    g = gray2.convert(gray2.init_timelike(0.7, xu8), gray2.BL)
    o = oracle.convert(oracle.init_timelike(0.7, xu8), oracle.BL)
    gray2.integrate(g, INF, gsc)
    oracle.integrate(o, INF, osc)
    gst = to_oracle_state(g)
    assert np.array_equal(gst.status, o.status) and np.array_equal(gst.nsteps, o.nsteps)
    live = o.status == oracle.MAXSTEPS
    assert live.mean() > 0.95
    assert state_rel_error_bl(gst.q[:, live], o.q[:, live]).max() < TOL_STATE_F64


# ---- stopping rule, resume, the singular axis ---------------------------------------------------------

def away_from_axis_pair(cfg):
    """The rays of an image that keep AXIS_MARGIN from the axis, as a GPU and an oracle BL state (explicit
    null 8-vectors through gray2_init_explicit, the way bench.py's end-to-end leg feeds rays)."""
    k0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    keep = np.where(ih.axis_approach(k0) >= AXIS_MARGIN)[0]
    xu8 = np.ascontiguousarray(k0.q[:, keep].T)
    g = gray2.init_explicit(k0.a_eff, xu8, gray2.NULL)
    o = oracle.init_explicit(k0.a_eff, xu8, oracle.NULL)
    return gray2.convert(g, gray2.BL), oracle.convert(o, oracle.BL)


def test_bl_resume_max_steps_and_lambda_end():
    cfg = inputs.CFG3_NULL.scaled(33, 29)
    gsc, osc = bl_sc(cfg)
    g, o = away_from_axis_pair(cfg)
    assert g.n > 0.9 * cfg.nx * cfg.ny
    for lam_end in (500.0, 1000.5, INF):
        stats = gray2.new_stats()
        gray2.integrate(g, lam_end, gsc, stats=stats)
        ostats = oracle.integrate(o, lam_end, osc)
        gst = to_oracle_state(g)
        same = (gst.status == o.status) & (gst.nsteps == o.nsteps)
        assert same.mean() > 0.99                    # all but near-critical rays
        esc = same & (o.status != oracle.CAPTURED)
        assert state_rel_error_bl(gst.q[:, esc], o.q[:, esc]).max() < TOL_STATE_F64
        assert state_rel_error_bl(gst.q[:, same], o.q[:, same]).max() < TOL_STATE_BL_CAPTURED
        if lam_end != INF:
            assert np.array_equal(gst.status, o.status) and np.array_equal(gst.nsteps, o.nsteps)
            assert gray2.stats_dict(stats) == ostats
            active = gst.status == gray2.ACTIVE
            assert active.sum() > 0.8 * g.n
            assert np.allclose(gst.lam[active], lam_end, rtol=0, atol=1e-9)
    before = g.clone()
    gray2.integrate(g, INF, gsc)                       # nothing ACTIVE any more: a no-op
    assert torch.equal(before.q, g.q) and torch.equal(before.nsteps, g.nsteps)
    gsc7, osc7 = bl_sc(cfg, max_steps=7)
    g7 = gray2.convert(gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny), gray2.BL)
    stats = gray2.new_stats()
    gray2.integrate(g7, INF, gsc7, stats=stats)
    assert (g7.status == gray2.MAXSTEPS).all() and (g7.nsteps == 7).all()
    assert gray2.stats_dict(stats)["steps"] == 7 * cfg.nx * cfg.ny


def test_bl_axis_is_singular_and_reported_as_data():
    """the poles are coordinate singularities of BL.  A ray that starts on the axis has no
    finite BL velocity: INVALID at the first test, never stepped, in the oracle and on the GPU alike; the
    same ray in Kerr-Schild coordinates integrates without any special handling."""
    xu8 = np.array([[0.0, 0.0, 0.0, 50.0, 1.2, 0.05, 0.0, -1.0]])
    g = gray2.init_timelike(0.5, xu8, renormalise_ut=True)
    o = oracle.init_timelike(0.5, xu8, renormalise_ut=True)
    gsc, osc = sc_pair(mode=1, eta=0.01, r_escape=100.0, max_steps=5000, capture_factor=BL_CAPTURE)
    gb, ob = gray2.convert(g, gray2.BL), oracle.convert(o, oracle.BL)
    stats = gray2.new_stats()
    gray2.integrate(gb, INF, gsc, stats=stats)
    ostats = oracle.integrate(ob, INF, osc)
    assert gb.status.item() == gray2.INVALID and ob.status[0] == oracle.INVALID
    assert gray2.stats_dict(stats) == ostats and ostats["steps"] == 0
    gray2.integrate(g, INF, gsc)
    oracle.integrate(o, INF, osc)
    assert g.status.item() == o.status[0] and g.status.item() in (gray2.CAPTURED, gray2.ESCAPED)


# ---- full size, in the launch configuration bench.py --form bl times ----------------------------------

@pytest.mark.parametrize("prec", [gray2.F64, gray2.F32], ids=["f64", "f32"])
def test_bl_full_size_cfg3_sampled_parity(prec):
    cfg = inputs.CFG3_NULL
    gsc, osc = bl_sc(cfg)
    ks = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
    g = gray2.convert(ks, gray2.BL)
    rng = np.random.default_rng(1706)
    idx = np.sort(rng.choice(cfg.n, 1536, replace=False))
    g0 = take(to_oracle_state(g), idx)                   # the sampled rays' initial BL state as the kernel reads it
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    gstats = gray2.stats_dict(stats)
    assert gstats["n_active"] == 0
    assert gstats["steps"] == int(g.nsteps.sum(dtype=torch.int64).item())
    full0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    k0 = take(full0, idx) if prec == gray2.F64 else take(to_oracle_state(ks), idx)
    o0 = oracle.convert(k0, oracle.BL) if prec == gray2.F64 else g0     # FP32: the same float inputs, widened
    o = o0.copy()
    oracle.integrate(o, INF, osc)
    gst = take(to_oracle_state(g), idx)
    xi, eta, _, _ = ih.ray_constants(k0)
    _, beta = ih.pixel_grid(cfg)
    a_inf, b_inf = ih.asymptotic_image_point(full0.a_eff, cfg.inclination, xi, eta, np.where(beta[idx] >= 0, 1.0, -1.0))
    d = ih.band_distance(cfg.a, cfg.inclination, a_inf, b_inf)
    away = ih.axis_approach(k0) >= AXIS_MARGIN
    mask = ih.potential_mask(full0.a_eff, xi, eta, 900.0)
    if prec == gray2.F64:
        outside = (d > 1e-3) & away
        assert np.array_equal(gst.status[outside], o.status[outside]) and np.array_equal(gst.nsteps[outside], o.nsteps[outside])
        err = state_rel_error_bl(gst.q[:, outside], o.q[:, outside])
        cap = (o.status == oracle.CAPTURED)[outside]
        assert err[~cap].max() < TOL_STATE_F64 and err[cap].max() < TOL_STATE_BL_CAPTURED
    else:
        kw = bl_sc_kw(cfg)
        sens = twin_sensitivity(k0, kw)
        outside, _ = assert_fp32_parity(cfg.name + " Boyer-Lindquist, full size, 1536 sampled rays", gst, o, sens,
                                        state_rel_error_bl(gst.q, o.q), bl_straddle_check(o0, gst, o, kw), usable=away,
                                        tol_scale=bl_fp32_tolerances(o))
    assert np.array_equal((gst.status == gray2.CAPTURED)[outside], mask[outside])
    # a property of the whole image: apart from the rays lost near the axis (DESIGN R21) the captured
    # fraction is the area of Bardeen's curve over the field of view
    ca, cb = __import__("closed_forms").bardeen_curve(cfg.a, cfg.inclination)
    order = np.argsort(ca)
    area = 2.0 * np.trapezoid(cb[order], ca[order])
    assert abs(gstats["n_captured"] / cfg.n - area / (2 * cfg.fov) ** 2) < 4e-3
    assert gstats["n_invalid"] + gstats["n_maxsteps"] < 2e-3 * cfg.n
