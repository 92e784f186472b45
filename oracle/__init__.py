"""CPU ORACLE for the GRay2 hot path -- TEST INFRASTRUCTURE ONLY.

A ctypes wrapper around ``oracle/gray2_oracle.c`` (plain C, double precision, written from
/root/reference/PAPER.md eq. (2)-(8) and the classic RK4 of PAPER.md:164).  It shares no code with
the CUDA path in ``paper_1706_07062_b200/`` and neither imports the other.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may import it.

Every array argument and result is a HOST numpy array.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gray2_oracle.c")
_HDR = os.path.join(_HERE, "gray2_oracle.h")
_LIB = os.path.join(_HERE, "liboracle_gray2.so")

ACTIVE, CAPTURED, ESCAPED, MAXSTEPS, INVALID = 0, 1, 2, 3, 4
NULL, TIMELIKE = 0, 1
KS, BL = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP).  Returns the path of the shared library."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", tmp, _SRC, "-lm"]
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


class _State(C.Structure):
    _fields_ = [("q", C.c_void_p * 8), ("lam", C.c_void_p), ("status", C.c_void_p),
                ("nsteps", C.c_void_p), ("n", C.c_uint64), ("a_eff", C.c_double),
                ("kind", C.c_int32), ("reversed", C.c_int32), ("coords", C.c_int32)]


class _StepControl(C.Structure):
    _fields_ = [("mode", C.c_int32), ("h_fixed", C.c_double), ("eta", C.c_double),
                ("dir", C.c_int32), ("capture_factor", C.c_double), ("r_escape", C.c_double),
                ("max_steps", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in
                ("steps", "n_captured", "n_escaped", "n_maxsteps", "n_invalid", "n_active")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        d, p = C.c_double, C.c_void_p
        _lib.oracle_ks_r.restype = d
        _lib.oracle_ks_r.argtypes = [d, d, d, d]
        for name in ("oracle_ks_metric", "oracle_ks_metric_inverse", "oracle_ks_dmetric",
                     "oracle_ks_christoffel"):
            getattr(_lib, name).argtypes = [d, p, p]
            getattr(_lib, name).restype = None
        _lib.oracle_ks_dmetric_fd.argtypes = [d, p, d, p]
        _lib.oracle_ks_accel.argtypes = [d, p, p, p]
        _lib.oracle_ks_accel_fd.argtypes = [d, p, p, d, p]
        _lib.oracle_rk4_step.argtypes = [d, p, d]
        _lib.oracle_invariants_one.argtypes = [d, C.c_int32, p, p]
        _lib.oracle_trajectory.argtypes = [d, p, d, C.c_int64, C.c_int64, p]
        _lib.oracle_bl_metric.argtypes = [d, p, p]
        _lib.oracle_bl_accel.argtypes = [d, p, p, p]
        _lib.oracle_bl_accel_fd.argtypes = [d, p, p, p]
        _lib.oracle_bl_dmetric.argtypes = [d, p, p]
        _lib.oracle_bl_dmetric_fd.argtypes = [d, p, p]
        _lib.oracle_bl_rk4_step.argtypes = [d, p, d]
        _lib.oracle_bl_rk4_step_guarded.argtypes = [d, p, d, d]
        _lib.oracle_bl_invariants_one.argtypes = [d, C.c_int32, p, p]
        _lib.oracle_bl_to_ks_one.argtypes = [d, p, p]
        _lib.oracle_ks_to_bl_one.argtypes = [d, p, p]
        _lib.oracle_convert.argtypes = [p, p, C.c_uint64, C.c_int32]
        _lib.oracle_bl_trajectory.argtypes = [d, p, d, C.c_int64, C.c_int64, p]
        _lib.oracle_init_null.argtypes = [p, d, d, d, d, d, C.c_int32, C.c_int32]
        _lib.oracle_init_timelike.argtypes = [p, d, p, C.c_uint64, C.c_int32]
        _lib.oracle_init_explicit.argtypes = [p, d, p, C.c_uint64, C.c_int32, C.c_int32]
        _lib.oracle_integrate.argtypes = [p, C.c_uint64, d, p, p]
        _lib.oracle_invariants.argtypes = [p, C.c_uint64, p, p, p, p]
        _lib.oracle_ks_coordtime_accel.argtypes = [d, p, p, p]
        _lib.oracle_rk4_step_coordtime.argtypes = [d, p, d]
        _lib.oracle_trajectory_coordtime.argtypes = [d, p, d, C.c_int64, C.c_int64, p]
        _lib.oracle_integrate_coordtime.argtypes = [p, C.c_uint64, d, p, p]
        _lib.oracle_integrate_diagnostics.argtypes = [p, C.c_uint64, d, p, p, p]
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _vec(v, n):
    a = np.ascontiguousarray(np.asarray(v, dtype=np.float64).reshape(-1))
    assert a.size == n, (a.size, n)
    return a


@dataclass
class State:
    """Host SoA state of n geodesics (same fields as gray2_state in include/gray2.h)."""
    n: int
    q: np.ndarray = field(default=None)        # (8, n) float64 : t,x,y,z,u^t,u^x,u^y,u^z (KS) or
                                               #                  t,r,theta,phi,u^t,u^r,u^theta,u^phi (BL)
    lam: np.ndarray = field(default=None)      # (n,) float64
    status: np.ndarray = field(default=None)   # (n,) int32
    nsteps: np.ndarray = field(default=None)   # (n,) int32
    a_eff: float = 0.0
    kind: int = NULL
    reversed: int = 0
    coords: int = KS

    def __post_init__(self):
        if self.q is None:
            self.q = np.zeros((8, self.n), dtype=np.float64)
            self.lam = np.zeros(self.n, dtype=np.float64)
            self.status = np.zeros(self.n, dtype=np.int32)
            self.nsteps = np.zeros(self.n, dtype=np.int32)

    def _c(self) -> _State:
        s = _State()
        for m in range(8):
            s.q[m] = self.q[m].ctypes.data
        s.lam = self.lam.ctypes.data
        s.status = self.status.ctypes.data
        s.nsteps = self.nsteps.ctypes.data
        s.n = self.n
        s.a_eff = self.a_eff
        s.kind = self.kind
        s.reversed = self.reversed
        s.coords = self.coords
        return s

    def _back(self, s: _State):
        self.a_eff, self.kind, self.reversed, self.coords = s.a_eff, s.kind, s.reversed, s.coords

    def copy(self) -> "State":
        return State(self.n, self.q.copy(), self.lam.copy(), self.status.copy(), self.nsteps.copy(),
                     self.a_eff, self.kind, self.reversed, self.coords)


def step_control(mode=1, h_fixed=0.0, eta=0.01, dir=1, capture_factor=1.01, r_escape=float("inf"),
                 max_steps=20000) -> _StepControl:
    return _StepControl(mode, h_fixed, eta, dir, capture_factor, r_escape, max_steps)


# ---- the four operations -------------------------------------------------------------------------

def init_null(a, r_obs, inclination_rad, fov_half_alpha, fov_half_beta, nx, ny) -> State:
    st = State(nx * ny)
    cs = st._c()
    rc = lib().oracle_init_null(C.byref(cs), a, r_obs, inclination_rad, fov_half_alpha,
                                fov_half_beta, nx, ny)
    if rc:
        raise ValueError("oracle_init_null: invalid arguments")
    st._back(cs)
    return st


def init_timelike(a, xu8, renormalise_ut=False) -> State:
    xu8 = np.ascontiguousarray(np.asarray(xu8, dtype=np.float64).reshape(-1, 8))
    st = State(xu8.shape[0])
    cs = st._c()
    rc = lib().oracle_init_timelike(C.byref(cs), a, _ptr(xu8), xu8.shape[0], int(renormalise_ut))
    if rc:
        raise ValueError("oracle_init_timelike: invalid arguments")
    st._back(cs)
    return st


def init_explicit(a, xu8, kind=NULL, renormalise_ut=False) -> State:
    """Explicit 8-vectors of null (Table 1) or time-like geodesics."""
    xu8 = np.ascontiguousarray(np.asarray(xu8, dtype=np.float64).reshape(-1, 8))
    st = State(xu8.shape[0])
    cs = st._c()
    rc = lib().oracle_init_explicit(C.byref(cs), a, _ptr(xu8), xu8.shape[0], int(kind), int(renormalise_ut))
    if rc:
        raise ValueError("oracle_init_explicit: invalid arguments")
    st._back(cs)
    return st


def integrate(st: State, lambda_end, sc: _StepControl, n=None) -> dict:
    cs = st._c()
    stats = _Stats()
    rc = lib().oracle_integrate(C.byref(cs), st.n if n is None else n, float(lambda_end),
                                C.byref(sc), C.byref(stats))
    if rc:
        raise ValueError("oracle_integrate: invalid arguments")
    return {k: int(getattr(stats, k)) for k, _ in _Stats._fields_}


def integrate_coordtime(st: State, t_end, sc: _StepControl, n=None) -> dict:
    """Coordinate-time form (eq. 15): see oracle_integrate_coordtime in gray2_oracle.h."""
    cs = st._c()
    stats = _Stats()
    rc = lib().oracle_integrate_coordtime(C.byref(cs), st.n if n is None else n, float(t_end),
                                          C.byref(sc), C.byref(stats))
    if rc:
        raise ValueError("oracle_integrate_coordtime: invalid arguments")
    return {k: int(getattr(stats, k)) for k, _ in _Stats._fields_}


def integrate_diagnostics(st: State, lambda_end, sc: _StepControl, n=None):
    """Integrate and accumulate the paper's convergence diagnostics.  Returns (stats, diag) with
    diag = dict(max_abs_u2, cos_peak, dphi_cycle, t_zmax1, t_zmax2), each (n,) float64 (NaN = never)."""
    n = st.n if n is None else n
    out = np.empty((5, n), dtype=np.float64)
    cs = st._c()
    stats = _Stats()
    rc = lib().oracle_integrate_diagnostics(C.byref(cs), n, float(lambda_end), C.byref(sc), _ptr(out), C.byref(stats))
    if rc:
        raise ValueError("oracle_integrate_diagnostics: invalid arguments")
    names = ("max_abs_u2", "cos_peak", "dphi_cycle", "t_zmax1", "t_zmax2")
    return {k: int(getattr(stats, k)) for k, _ in _Stats._fields_}, dict(zip(names, out))


def invariants(st: State):
    """Returns E, Lz, Q, norm (each (n,) float64) of the RUN geodesic (see gray2.h sign rule)."""
    out = [np.empty(st.n, dtype=np.float64) for _ in range(4)]
    cs = st._c()
    rc = lib().oracle_invariants(C.byref(cs), st.n, *[_ptr(o) for o in out])
    if rc:
        raise ValueError("oracle_invariants: invalid arguments")
    return tuple(out)


# ---- building blocks -----------------------------------------------------------------------------

def ks_r(a, x, y, z) -> float:
    return lib().oracle_ks_r(a, x, y, z)


def _mat(fn, a, pos, n_out, shape):
    pos = _vec(pos, 3)
    out = np.empty(n_out, dtype=np.float64)
    fn(a, _ptr(pos), _ptr(out))
    return out.reshape(shape)


def ks_metric(a, pos):
    return _mat(lib().oracle_ks_metric, a, pos, 16, (4, 4))


def ks_metric_inverse(a, pos):
    return _mat(lib().oracle_ks_metric_inverse, a, pos, 16, (4, 4))


def ks_dmetric(a, pos):
    """dg[c, a, b] = d_c g_ab (analytic)."""
    return _mat(lib().oracle_ks_dmetric, a, pos, 64, (4, 4, 4))


def ks_dmetric_fd(a, pos, step=1e-5):
    pos = _vec(pos, 3)
    out = np.empty(64, dtype=np.float64)
    lib().oracle_ks_dmetric_fd(a, _ptr(pos), step, _ptr(out))
    return out.reshape(4, 4, 4)


def ks_christoffel(a, pos):
    """Gam[m, a, b] = Gamma^m_ab."""
    return _mat(lib().oracle_ks_christoffel, a, pos, 64, (4, 4, 4))


def ks_accel(a, pos, u):
    pos, u = _vec(pos, 3), _vec(u, 4)
    out = np.empty(4, dtype=np.float64)
    lib().oracle_ks_accel(a, _ptr(pos), _ptr(u), _ptr(out))
    return out


def ks_accel_fd(a, pos, u, step=1e-5):
    pos, u = _vec(pos, 3), _vec(u, 4)
    out = np.empty(4, dtype=np.float64)
    lib().oracle_ks_accel_fd(a, _ptr(pos), _ptr(u), step, _ptr(out))
    return out


def rk4_step(a, y, h):
    y = _vec(y, 8).copy()
    lib().oracle_rk4_step(a, _ptr(y), h)
    return y


def invariants_one(a, kind, y):
    y = _vec(y, 8)
    out = np.empty(4, dtype=np.float64)
    lib().oracle_invariants_one(a, kind, _ptr(y), _ptr(out))
    return out


def trajectory(a, y0, h, nsteps, stride=1):
    y0 = _vec(y0, 8)
    out = np.empty((nsteps // stride + 1, 8), dtype=np.float64)
    lib().oracle_trajectory(a, _ptr(y0), h, nsteps, stride, _ptr(out))
    return out


def ks_coordtime_accel(a, pos, v):
    pos, v = _vec(pos, 3), _vec(v, 3)
    out = np.empty(3, dtype=np.float64)
    lib().oracle_ks_coordtime_accel(a, _ptr(pos), _ptr(v), _ptr(out))
    return out


def trajectory_coordtime(a, y0, h, nsteps, stride=1):
    """y0 = (t,x,y,z,vx,vy,vz); rows of the result likewise."""
    y0 = _vec(y0, 7)
    out = np.empty((nsteps // stride + 1, 7), dtype=np.float64)
    lib().oracle_trajectory_coordtime(a, _ptr(y0), h, nsteps, stride, _ptr(out))
    return out


def bl_metric(a, X):
    X = _vec(X, 4)
    out = np.empty(16, dtype=np.float64)
    lib().oracle_bl_metric(a, _ptr(X), _ptr(out))
    return out.reshape(4, 4)


def bl_accel(a, X, u):
    X, u = _vec(X, 4), _vec(u, 4)
    out = np.empty(4, dtype=np.float64)
    lib().oracle_bl_accel(a, _ptr(X), _ptr(u), _ptr(out))
    return out


def bl_accel_fd(a, X, u):
    X, u = _vec(X, 4), _vec(u, 4)
    out = np.empty(4, dtype=np.float64)
    lib().oracle_bl_accel_fd(a, _ptr(X), _ptr(u), _ptr(out))
    return out


def bl_dmetric(a, X, fd=False):
    """dg[c, a, b] = d_c g_ab of PAPER.md eq. (1); fd=True: 4th-order central differences of bl_metric."""
    X = _vec(X, 4)
    out = np.empty(64, dtype=np.float64)
    (lib().oracle_bl_dmetric_fd if fd else lib().oracle_bl_dmetric)(a, _ptr(X), _ptr(out))
    return out.reshape(4, 4, 4)


def bl_rk4_step(a, y, h):
    y = _vec(y, 8).copy()
    lib().oracle_bl_rk4_step(a, _ptr(y), h)
    return y


def bl_rk4_step_guarded(a, y, h, r_capture):
    """(violated, y_new): y_new == y when a stage position had r < r_capture."""
    y = _vec(y, 8).copy()
    rc = lib().oracle_bl_rk4_step_guarded(a, _ptr(y), h, r_capture)
    return bool(rc), y


def bl_invariants_one(a, kind, y):
    y = _vec(y, 8)
    out = np.empty(4, dtype=np.float64)
    lib().oracle_bl_invariants_one(a, kind, _ptr(y), _ptr(out))
    return out


def bl_to_ks_one(a, y):
    y = _vec(y, 8)
    out = np.empty(8, dtype=np.float64)
    lib().oracle_bl_to_ks_one(a, _ptr(y), _ptr(out))
    return out


def ks_to_bl_one(a, y):
    y = _vec(y, 8)
    out = np.empty(8, dtype=np.float64)
    lib().oracle_ks_to_bl_one(a, _ptr(y), _ptr(out))
    return out


def convert(st: State, to_coords: int, n=None) -> State:
    """A new State in the other coordinate system (KS <-> BL), same geodesics."""
    n = st.n if n is None else n
    out = State(st.n)
    cs, cd = st._c(), out._c()
    rc = lib().oracle_convert(C.byref(cs), C.byref(cd), n, to_coords)
    if rc != 0:
        raise ValueError("oracle_convert: bad arguments")
    out._back(cd)
    return out


def bl_trajectory(a, y0, h, nsteps, stride=1):
    y0 = _vec(y0, 8)
    out = np.empty((nsteps // stride + 1, 8), dtype=np.float64)
    lib().oracle_bl_trajectory(a, _ptr(y0), h, nsteps, stride, _ptr(out))
    return out


def num_threads() -> int:
    return int(lib().oracle_num_threads())
