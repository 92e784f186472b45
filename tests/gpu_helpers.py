"""Helpers for the GPU parity tests: run a config through the C-ABI binding and through the oracle and
compare element by element with the tolerances BASELINE.json's north_star states.

Tolerances (written here once, used by every parity test):
  FP64  final 8-vector: relative 1e-9 w.r.t. max(|component|, r), for rays with identical step counts
        capture/escape flag and nsteps: bit-exact outside the critical band (d > 1e-3 M, DESIGN R11)
        invariant drift (end - start): equal to the oracle's within 1e-12 of the size of the terms the
        invariant is a sum of at the final state: E ~ u^t, L_z ~ R|v|, Q ~ (R|v|)^2, norm ~ (u^t)^2
        (at r ~ 1100 the terms of Q are ~1e6 and cancel to ~30, so 1e-12 of |Q| is below its rounding)
  FP32  final 8-vector: relative 1e-4, rays with identical step counts, outside the band
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


def image_sc(cfg):
    return sc_pair(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                   capture_factor=cfg.capture_factor)


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
