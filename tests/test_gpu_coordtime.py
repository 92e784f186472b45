"""GPU parity of the coordinate-time form (gray2_integrate_coordtime) against the
oracle's literal eq. (15), element by element, plus its edge cases."""
import numpy as np
import pytest
import torch

import image_helpers as ih
import oracle
from gpu_helpers import (INF, TOL_STATE_F32, TOL_STATE_F64, assert_fp32_parity, image_sc, image_sc_kw, make_straddle_check,
                         sc_pair, state_rel_error, take, to_oracle_state, twin_sensitivity)
from paper_1706_07062_b200 import gray2, inputs

pytestmark = pytest.mark.gpu


def test_timelike_ensemble_to_a_target_time():
    xu8, _ = inputs.cfg4_ensemble(3001)         # several blocks and a ragged tail
    gsc, osc = sc_pair(mode=0, h_fixed=0.7, max_steps=100000)
    g = gray2.init_timelike(0.7, xu8)
    o = oracle.init_timelike(0.7, xu8)
    stats = gray2.new_stats()
    gray2.integrate_coordtime(g, 500.0, gsc, stats=stats)
    ostats = oracle.integrate_coordtime(o, 500.0, osc)
    gst = to_oracle_state(g)
    assert gray2.stats_dict(stats) == ostats
    assert (gst.status == gray2.ACTIVE).all() and np.array_equal(gst.nsteps, o.nsteps) and (gst.nsteps == 715).all()
    assert np.allclose(gst.q[0], 500.0, atol=1e-10) and (gst.q[4] == 1.0).all()
    assert (g.lam == 0).all()                                        # lambda is not touched
    assert state_rel_error(gst.q, o.q, 0.7).max() < TOL_STATE_F64
    # resume to a later target, against the oracle resumed the same way; a second call is a no-op
    gray2.integrate_coordtime(g, 800.0, gsc, stats=stats)
    oracle.integrate_coordtime(o, 800.0, osc)
    gst = to_oracle_state(g)
    assert np.array_equal(gst.nsteps, o.nsteps) and state_rel_error(gst.q, o.q, 0.7).max() < TOL_STATE_F64
    snap = g.q.clone()
    gray2.integrate_coordtime(g, 800.0, gsc, stats=stats)
    assert gray2.stats_dict(stats)["steps"] == 0 and torch.equal(snap, g.q)


@pytest.mark.parametrize("cfg", [inputs.CFG1_NULL, inputs.CFG3_NULL.scaled(97, 61)], ids=lambda c: c.name)
def test_null_images_in_coordinate_time(cfg):
    """Same rays, stepped in t with dt = eta r: status and step counts exact outside the band, states 1e-9,
    and the same capture mask as Carter's potential."""
    gsc, osc = image_sc(cfg)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o = o0.copy()
    stats = gray2.new_stats()
    gray2.integrate_coordtime(g, INF, gsc, stats=stats)
    ostats = oracle.integrate_coordtime(o, INF, osc)
    gst = to_oracle_state(g)
    d, mask = ih.classify_image(cfg, o0)
    outside = d > 1e-3
    assert outside.mean() > 0.99
    assert np.array_equal(gst.status[outside], o.status[outside]) and np.array_equal(gst.nsteps[outside], o.nsteps[outside])
    assert np.array_equal((gst.status == gray2.CAPTURED)[outside], mask[outside])
    assert state_rel_error(gst.q[:, outside], o.q[:, outside], o.a_eff).max() < TOL_STATE_F64
    sd = gray2.stats_dict(stats)
    assert sd["n_active"] == 0 and sd["n_invalid"] == 0 and abs(sd["steps"] - ostats["steps"]) <= 60 * (~outside).sum()
    # the stored tangent (1, v) is null, and xi = Lz/E, eta = Q/E^2 are those of the initial ray
    E, Lz, Q, norm = [t.cpu().numpy() for t in gray2.invariants(g)]
    xi0, eta0, _, _ = ih.ray_constants(o0)
    esc = (gst.status == gray2.ESCAPED) & outside
    assert np.abs(norm / E ** 2)[esc].max() < 1e-5
    assert np.abs(Lz / E - xi0)[esc].max() < 1e-4 and np.abs(Q / E ** 2 - eta0)[esc].max() < 1e-3


def test_coordinate_time_fp32_and_edges():
    cfg = inputs.CFG3_NULL.scaled(64)
    gsc, osc = image_sc(cfg)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=gray2.F32)
    o0 = to_oracle_state(g)                              # the same inputs: the float initial state, widened
    o = o0.copy()
    gray2.integrate_coordtime(g, INF, gsc)
    oracle.integrate_coordtime(o, INF, osc)
    gst = to_oracle_state(g)
    kw = image_sc_kw(cfg)
    sens = twin_sensitivity(o0, kw)                      # a property of the geodesic: measured on the affine run
    noncrit, same = assert_fp32_parity(cfg.name + " coordinate time", gst, o, sens, state_rel_error(gst.q, o.q, o.a_eff),
                                       make_straddle_check(o0, gst, o, kw, driver=oracle.integrate_coordtime))
    xi, eta, _, _ = ih.ray_constants(o0)
    mask = ih.potential_mask(o0.a_eff, xi, eta, 0.9 * cfg.r_obs)
    assert np.array_equal((gst.status == gray2.CAPTURED)[noncrit], mask[noncrit])
    # INVALID input, tiny batch, max_steps
    xu8, _ = inputs.cfg4_ensemble(5)
    xu8[2, 0] = np.nan
    g2 = gray2.init_timelike(0.7, xu8)
    stats = gray2.new_stats()
    gray2.integrate_coordtime(g2, INF, gray2.step_control(mode=0, h_fixed=0.5, max_steps=40), stats=stats)
    sd = gray2.stats_dict(stats)
    assert sd["n_invalid"] == 1 and sd["n_maxsteps"] == 4 and sd["steps"] == 160
    assert g2.status[2].item() == gray2.INVALID and g2.nsteps[2].item() == 0
    o2 = oracle.init_timelike(0.7, xu8)
    ostats = oracle.integrate_coordtime(o2, INF, oracle.step_control(mode=0, h_fixed=0.5, max_steps=40))
    assert ostats == sd


def test_backward_in_coordinate_time_retraces():
    xu8, _ = inputs.cfg4_ensemble(64)
    g = gray2.init_timelike(0.7, xu8)
    v0 = xu8[:, 5:8] / xu8[:, 4:5]
    gray2.integrate_coordtime(g, 60.0, gray2.step_control(mode=0, h_fixed=0.25, max_steps=10 ** 6))
    gray2.integrate_coordtime(g, 0.0, gray2.step_control(mode=0, h_fixed=0.25, dir=-1, max_steps=10 ** 6))
    q = g.q.cpu().numpy()
    assert np.abs(q[0]).max() < 1e-12 and np.abs(q[1:4] - xu8[:, 1:4].T).max() < 1e-6
    assert np.abs(q[5:8] - v0.T).max() < 1e-7
