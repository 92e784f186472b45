"""Helpers for the GPU parity tests: run a config through the C-ABI binding and through the oracle and
compare element by element with the tolerances BASELINE.json's north_star states.

Tolerances (written here once, used by every parity test):
  FP64  final 8-vector: relative 1e-9 w.r.t. max(|component|, r), for rays with identical step counts
        capture/escape flag and nsteps: bit-exact outside the critical band (d > 1e-3 M, DESIGN R11)
        invariant drift (end - start): equal to the oracle's within 1e-12 of the size of the terms the
        invariant is a sum of at the final state: E ~ u^t, L_z ~ R|v|, Q ~ (R|v|)^2, norm ~ (u^t)^2
        (at r ~ 1100 the terms of Q are ~1e6 and cancel to ~30, so 1e-12 of |Q| is below its rounding)
  FP32  final 8-vector, all eight components: relative 1e-4 on EVERY non-critical ray, the oracle being given
        the float initial state; non-critical = final state stable to 1e-4 under one FP32 rounding error of the
        starting point (twin rays, oracle only; see "FP32 parity" below and DESIGN R12)
"""
import numpy as np
import torch

import oracle
from paper_1706_07062_b200 import build as _build
from paper_1706_07062_b200 import gray2

_build.build()   # in-tree nvcc build; a no-op when libgray2.so is newer than its sources

INF = float("inf")
TOL_STATE_F64 = 1e-9
TOL_STATE_F32 = 1e-4
TOL_DRIFT_F64 = 1e-12


def to_oracle_state(st: gray2.State) -> oracle.State:
    """Copy a device state to a host oracle.State (float32 states are widened)."""
    return oracle.State(st.n, st.q.double().cpu().numpy().copy(), st.lam.cpu().numpy().copy(),
                        st.status.cpu().numpy().copy(), st.nsteps.cpu().numpy().copy(),
                        st.a_eff, st.kind, st.reversed, st.coords)


def sc_pair(**kw):
    return gray2.step_control(**kw), oracle.step_control(**kw)


def image_sc_kw(cfg):
    return dict(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps, capture_factor=cfg.capture_factor)


def image_sc(cfg):
    return sc_pair(**image_sc_kw(cfg))


def run_gpu_image(cfg, prec=gray2.F64):
    st = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
    st0 = st.clone()
    stats = gray2.new_stats()
    gray2.integrate(st, INF, image_sc(cfg)[0], stats=stats)
    torch.cuda.synchronize()
    return st0, st, gray2.stats_dict(stats)


def run_oracle_image(cfg, subset=None):
    st0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    if subset is not None:
        st0 = take(st0, subset)
    st = st0.copy()
    stats = oracle.integrate(st, INF, image_sc(cfg)[1])
    return st0, st, stats


def take(st: oracle.State, idx) -> oracle.State:
    idx = np.asarray(idx)
    return oracle.State(len(idx), np.ascontiguousarray(st.q[:, idx]), st.lam[idx].copy(), st.status[idx].copy(),
                        st.nsteps[idx].copy(), st.a_eff, st.kind, st.reversed, st.coords)


def state_rel_error(gq: np.ndarray, oq: np.ndarray, a_eff: float) -> np.ndarray:
    """max over the 8 components of |gpu - oracle| / max(|oracle component|, r), per ray."""
    r = np.array([oracle.ks_r(a_eff, oq[1, k], oq[2, k], oq[3, k]) for k in range(oq.shape[1])])
    scale = np.maximum(np.abs(oq), r[None, :])
    return np.max(np.abs(gq - oq) / scale, axis=0)


def state_rel_error_bl(gq: np.ndarray, oq: np.ndarray) -> np.ndarray:
    """The same measure for Boyer-Lindquist states (t, r, theta, phi, and their derivatives): lengths
    relative to max(|component|, r), angles to max(|angle|, 1), angular velocities to max(|.|, 1/r)."""
    r = np.abs(oq[1])
    one = np.ones_like(r)
    scale = np.stack([np.maximum(np.abs(oq[0]), r), r, np.maximum(np.abs(oq[2]), one), np.maximum(np.abs(oq[3]), one),
                      np.maximum(np.abs(oq[4]), one), np.maximum(np.abs(oq[5]), one),
                      np.maximum(np.abs(oq[6]), 1.0 / r), np.maximum(np.abs(oq[7]), 1.0 / r)])
    return np.max(np.abs(gq - oq) / scale, axis=0)


def drift(inv_end, inv_start):
    return [e - s for e, s in zip(inv_end, inv_start)]


def gpu_invariants_np(st: gray2.State):
    return [t.cpu().numpy() for t in gray2.invariants(st)]


def invariant_term_scales(q: np.ndarray):
    """Size of the terms each invariant is a sum of (E, Lz, Q, norm), from an (8, n) state array."""
    R = np.sqrt((q[1:4] ** 2).sum(0))
    V = np.sqrt((q[5:8] ** 2).sum(0))
    ut = np.abs(q[4])
    return [np.maximum(1.0, ut), np.maximum(1.0, R * V), np.maximum(1.0, (R * V) ** 2), np.maximum(1.0, ut * ut)]


# ---- FP32 parity (DESIGN R12) -------------------------------------------------------------------------
# north_star: "final states must agree to relative ... 1e-4 in FP32 for non-critical rays after identical step
# sequences".  The oracle is given the SAME inputs as the FP32 kernel: the float initial state, widened.  Which
# rays are non-critical in FP32 is decided by the oracle alone, from the geodesic itself: a ray is critical when
# its final state moves by more than the tolerance when its initial data move by one FP32 rounding error: the
# starting point by half an ulp of its largest coordinate (3.05e-5 M for 512 <= |x| < 1024, the image plane at
# 1000 M), or the spatial velocity by half an ulp of its largest component (3e-8: the same 3e-5 M of impact
# parameter over the 1000 M to the hole) -- no FP32 computation can be asked to resolve such a ray, its input is
# not known better than that.  The sensitivity is measured with twin rays (two transverse directions each for
# position and velocity -- along the ray a displacement only relabels the affine parameter --, u^t re-solved, the
# same number of steps as the undisplaced ray).
def half_ulp_f32(x: np.ndarray) -> np.ndarray:
    return 0.5 * np.spacing(np.abs(x).astype(np.float32)).astype(np.float64)


def _fixed_count_run(st0: oracle.State, nsteps: np.ndarray, sc_kw: dict) -> oracle.State:
    """Every ray of st0 advanced by exactly nsteps[k] steps of the step rule in sc_kw, no stopping test."""
    big = int(nsteps.max()) + 1
    st = st0.copy()
    st.nsteps[:] = big - nsteps                      # max_steps counts from the state's nsteps
    kw = dict(sc_kw)
    kw.update(max_steps=big, r_escape=INF, capture_factor=1e-9)
    oracle.integrate(st, INF, oracle.step_control(**kw))
    return st


TWINS_TRANSVERSE = (("pos", "e1"), ("pos", "e2"), ("vel", "e1"), ("vel", "e2"))
# bound orbits run for many periods: what grows is the phase, driven by the energy (speed along the velocity) and
# by the angular momentum (velocity across it)
TWINS_ORBIT = (("vel", "v"), ("vel", "e1"), ("vel", "e2"), ("pos", "e1"))


def twin_sensitivity(k0: oracle.State, sc_kw: dict, rel_delta=None, twins=TWINS_TRANSVERSE) -> np.ndarray:
    """Per ray of the Kerr-Schild initial state k0: the largest relative change of the final state (the measure
    of state_rel_error, all eight components) when the starting point, or the spatial velocity, is displaced across
    the ray by half an FP32 ulp of its largest component (by rel_delta times its largest component when rel_delta
    is given), at a fixed number of steps.  Oracle only."""
    ref = k0.copy()
    oracle.integrate(ref, INF, oracle.step_control(**sc_kw))
    base = _fixed_count_run(k0, ref.nsteps, sc_kw)
    v = k0.q[5:8].T
    ez = np.broadcast_to(np.array([0.0, 0.0, 1.0]), v.shape)
    e1 = np.cross(v, ez)
    thin = np.linalg.norm(e1, axis=1) < 1e-6 * np.linalg.norm(v, axis=1)
    e1[thin] = np.cross(v[thin], np.array([1.0, 0.0, 0.0]))
    e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
    e2 = np.cross(v, e1)
    e2 /= np.linalg.norm(e2, axis=1, keepdims=True)
    sens = np.zeros(k0.n)
    direction = {"e1": e1, "e2": e2, "v": v / np.linalg.norm(v, axis=1, keepdims=True)}
    for what, along in twins:
        first = 1 if what == "pos" else 5
        big = np.abs(k0.q[first:first + 3]).max(axis=0)
        delta = half_ulp_f32(big) if rel_delta is None else rel_delta * big
        xu8 = np.ascontiguousarray(k0.q.T.copy())
        xu8[:, first:first + 3] += delta[:, None] * direction[along]
        tw0 = oracle.init_explicit(k0.a_eff, xu8, k0.kind, renormalise_ut=True)
        tw = _fixed_count_run(tw0, ref.nsteps, sc_kw)
        sens = np.maximum(sens, state_rel_error(tw.q, base.q, k0.a_eff))
    return sens


def assert_fp32_parity(label, gst: oracle.State, o: oracle.State, sens: np.ndarray, err: np.ndarray,
                       straddles, usable=None, tol=TOL_STATE_F32, tol_scale=None, min_noncrit=0.9):
    """The FP32 acceptance: on EVERY non-critical ray (sens <= tol; `usable` removes rays a test excludes for a
    stated reason, e.g. the Boyer-Lindquist axis) the status equals the oracle's, the step count equals the
    oracle's unless the ray straddles a stopping threshold (straddles(k) -> bool, checked with the oracle), and
    all eight components of the final state, t included, agree to `tol` (times tol_scale[k] where a test states
    a reason for a per-ray factor).  Prints how many rays were excluded."""
    if tol_scale is not None:
        err = err / tol_scale
    noncrit = sens <= tol
    if usable is not None:
        noncrit &= usable
    n_excl = int((~noncrit).sum())
    print("[fp32 parity] %s: %d of %d rays critical or excluded (%.2f %%), largest sensitivity kept %.2e"
          % (label, n_excl, gst.n, 100.0 * n_excl / gst.n, sens[noncrit].max() if noncrit.any() else 0.0))
    assert noncrit.mean() > min_noncrit, noncrit.mean()
    assert np.array_equal(gst.status[noncrit], o.status[noncrit])
    differ = np.flatnonzero(noncrit & (gst.nsteps != o.nsteps))
    assert len(differ) <= max(2, 1e-3 * gst.n), len(differ)
    for k in differ:
        assert abs(int(gst.nsteps[k]) - int(o.nsteps[k])) == 1 and straddles(k), (k, gst.nsteps[k], o.nsteps[k])
    same = noncrit & (gst.nsteps == o.nsteps)
    worst = err[same].max()
    print("[fp32 parity] %s: max error over %d rays %.2e (median %.2e), %d threshold straddlers"
          % (label, same.sum(), worst, np.median(err[same]), len(differ)))
    assert worst < tol, worst
    return noncrit, same


def make_straddle_check(o0: oracle.State, gst: oracle.State, o: oracle.State, sc_kw: dict, driver=None, rel=2e-5):
    """straddles(k): the stopping test that decided ray k was within FP32 rounding of its threshold: at the
    smaller of the two step counts the oracle's r is within `rel` of r_escape or of the capture radius."""
    r_plus = 1.0 + np.sqrt(1.0 - o0.a_eff ** 2)
    thresholds = (sc_kw.get("r_escape", INF), sc_kw.get("capture_factor", 1.01) * r_plus)

    def straddles(k):
        n = min(int(gst.nsteps[k]), int(o.nsteps[k]))
        one = take(o0, [k])
        kw = dict(sc_kw)
        kw.update(max_steps=n, r_escape=INF, capture_factor=1e-9)
        (driver or oracle.integrate)(one, INF, oracle.step_control(**kw))
        r = one.q[1, 0] if one.coords == oracle.BL else oracle.ks_r(one.a_eff, *one.q[1:4, 0])
        return any(np.isfinite(t) and abs(r / t - 1.0) < rel for t in thresholds)
    return straddles


def accumulated_rounding_f64(nsteps: int) -> float:
    """The relative perturbation a double-precision integration of nsteps RK4 steps is equivalent to: an error of
    one ulp, 2^-52, per right-hand-side evaluation (each is about a hundred rounded operations; neither side's result
    is better than that), 4 nsteps of them, accumulating like a random walk.  Two correct
    double implementations that round in different orders (the oracle's connection form, the kernel's regrouped
    form) differ by about this much in their effective initial data; an orbit whose final state moves by more than
    the tolerance under a perturbation of this size is critical in FP64 in the sense of north_star."""
    return 2.0 ** -52 * np.sqrt(4.0 * nsteps)
