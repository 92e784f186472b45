"""Thin Python binding of the C-ABI library ``libgray2.so`` (include/gray2.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of ``csrc/``.  PyTorch is
used for device memory and streams, nothing else.  There is no CPU fallback: if the library is not
built, or there is no CUDA device, the calls raise.

Function names match the C entry points: ``init_null``, ``init_explicit`` / ``init_timelike``,
``integrate``, ``invariants`` (plus the diagnostic ``rhs``).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

F64, F32 = 0, 1
NULL, TIMELIKE = 0, 1
KS, BL = 0, 1
ACTIVE, CAPTURED, ESCAPED, MAXSTEPS, INVALID = 0, 1, 2, 3, 4
OK, EINVAL, ESTATE, ECUDA = 0, 1, 2, 3

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgray2.so")


class Gray2Error(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("gray2 error %d: %s" % (code, msg))
        self.code = code


class _CState(C.Structure):
    _fields_ = [("q", C.c_void_p * 8), ("lam", C.c_void_p), ("status", C.c_void_p), ("nsteps", C.c_void_p),
                ("n", C.c_uint64), ("a_eff", C.c_double), ("prec", C.c_int32), ("kind", C.c_int32),
                ("reversed", C.c_int32), ("coords", C.c_int32), ("order", C.c_void_p)]


class StepControl(C.Structure):
    """gray2_step_control (see include/gray2.h)."""
    _fields_ = [("mode", C.c_int32), ("h_fixed", C.c_double), ("eta", C.c_double), ("dir", C.c_int32),
                ("capture_factor", C.c_double), ("r_escape", C.c_double), ("max_steps", C.c_int32)]


def step_control(mode=1, h_fixed=0.0, eta=0.01, dir=1, capture_factor=1.01, r_escape=float("inf"),
                 max_steps=20000) -> StepControl:
    return StepControl(mode, h_fixed, eta, dir, capture_factor, r_escape, max_steps)


STATS_FIELDS = ("steps", "n_captured", "n_escaped", "n_maxsteps", "n_invalid", "n_active")

_lib = None


def load_library():
    """Load libgray2.so.  Raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libgray2.so is missing: run `python -m paper_1706_07062_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    d, p, i32, u64 = C.c_double, C.c_void_p, C.c_int32, C.c_uint64
    lib.gray2_init_null.argtypes = [p, d, d, d, d, d, i32, i32, p]
    lib.gray2_init_timelike.argtypes = [p, d, p, u64, i32, p]
    lib.gray2_init_explicit.argtypes = [p, d, p, u64, i32, i32, p]
    lib.gray2_init_explicit.restype = C.c_int
    lib.gray2_init_explicit_noalloc.argtypes = [p, d, p, u64, i32, i32, p]
    lib.gray2_init_explicit_noalloc.restype = C.c_int
    lib.gray2_init_null_shard.argtypes = [p, d, d, d, d, d, i32, i32, u64, i32, i32, p]
    lib.gray2_shard_count.argtypes = [u64, u64, i32, i32]
    lib.gray2_shard_count.restype = u64
    lib.gray2_integrate.argtypes = [p, u64, d, p, i32, p, p]
    lib.gray2_integrate_coordtime.argtypes = [p, u64, d, p, i32, p, p]
    lib.gray2_integrate_coordtime.restype = C.c_int
    lib.gray2_flops_per_step_coordtime.argtypes = [i32]
    lib.gray2_flops_per_step_coordtime.restype = C.c_int
    lib.gray2_invariants.argtypes = [p, u64, p, p, p, p, p]
    lib.gray2_integrate_diagnostics.argtypes = [p, u64, d, p, i32, p, p, p]
    lib.gray2_integrate_diagnostics.restype = C.c_int
    lib.gray2_rhs.argtypes = [i32, d, u64, p, p, p, p]
    lib.gray2_rhs_bl.argtypes = [i32, d, u64, p, p, p, p]
    lib.gray2_convert.argtypes = [p, p, u64, i32, p]
    lib.gray2_flops_per_step_bl.argtypes = [i32]
    lib.gray2_set_launch.argtypes = [i32, i32, i32]
    lib.gray2_order_longest_first.argtypes = [p, u64, p, p]
    lib.gray2_order_longest_first.restype = C.c_int
    lib.gray2_flops_per_step.argtypes = [i32]
    for name in ("gray2_init_null", "gray2_init_timelike", "gray2_integrate", "gray2_invariants", "gray2_rhs",
                 "gray2_set_launch", "gray2_flops_per_step"):
        getattr(lib, name).restype = C.c_int
    lib.gray2_last_error.restype = C.c_char_p
    lib.gray2_version.restype = C.c_char_p
    _lib = lib
    return lib


def _check(rc):
    if rc != OK:
        raise Gray2Error(rc, load_library().gray2_last_error().decode())


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("gray2 needs a CUDA device (there is no CPU fallback)")


@dataclass
class State:
    """Device SoA state of n geodesics; the tensors are owned here and borrowed by the library."""
    n: int
    prec: int
    q: torch.Tensor          # (8, n) float64 or float32, cuda: t,x,y,z,u^t,u^x,u^y,u^z (KS) or
                             # t,r,theta,phi,u^t,u^r,u^theta,u^phi (BL)
    lam: torch.Tensor        # (n,) float64
    status: torch.Tensor     # (n,) int32
    nsteps: torch.Tensor     # (n,) int32
    a_eff: float = 0.0
    kind: int = NULL
    reversed: int = 0
    coords: int = KS
    order: torch.Tensor | None = None     # optional (n,) int32 cuda: the schedule of the integrators (gray2.h)

    @staticmethod
    def empty(n: int, prec: int = F64, device="cuda") -> "State":
        _require_cuda()
        dt = torch.float64 if prec == F64 else torch.float32
        return State(n, prec, torch.empty((8, n), dtype=dt, device=device),
                     torch.empty(n, dtype=torch.float64, device=device),
                     torch.empty(n, dtype=torch.int32, device=device),
                     torch.empty(n, dtype=torch.int32, device=device))

    def _c(self) -> _CState:
        s = _CState()
        for m in range(8):
            s.q[m] = self.q[m].data_ptr()
        s.lam, s.status, s.nsteps = self.lam.data_ptr(), self.status.data_ptr(), self.nsteps.data_ptr()
        s.n, s.a_eff, s.prec, s.kind, s.reversed = self.n, self.a_eff, self.prec, self.kind, self.reversed
        s.coords = self.coords
        if self.order is not None:
            assert self.order.is_cuda and self.order.dtype == torch.int32 and self.order.numel() == self.n
            assert self.order.is_contiguous() and self.order.device == self.q.device
            s.order = self.order.data_ptr()
        return s

    def _back(self, s: _CState):
        self.a_eff, self.kind, self.reversed, self.coords = s.a_eff, s.kind, s.reversed, s.coords

    def clone(self) -> "State":
        return State(self.n, self.prec, self.q.clone(), self.lam.clone(), self.status.clone(),
                     self.nsteps.clone(), self.a_eff, self.kind, self.reversed, self.coords, self.order)


def init_null(a, r_obs, inclination_rad, fov_half_alpha, fov_half_beta, nx, ny, prec=F64, stream=None,
              out: State | None = None) -> State:
    st = out if out is not None else State.empty(nx * ny, prec)
    cs = st._c()
    _check(load_library().gray2_init_null(C.byref(cs), a, r_obs, inclination_rad, fov_half_alpha,
                                          fov_half_beta, nx, ny, _stream_ptr(stream)))
    st._back(cs)
    return st


def shard_count(n, tile_rays, rank, world) -> int:
    return int(load_library().gray2_shard_count(n, tile_rays, rank, world))


def init_null_shard(a, r_obs, inclination_rad, fov_half_alpha, fov_half_beta, nx, ny, tile_rays, rank, world,
                    prec=F64, stream=None, out: State | None = None) -> State:
    """This rank's rays of an image dealt out in tiles of tile_rays to `world` GPUs (see gray2.h)."""
    st = out if out is not None else State.empty(shard_count(nx * ny, tile_rays, rank, world), prec)
    cs = st._c()
    _check(load_library().gray2_init_null_shard(C.byref(cs), a, r_obs, inclination_rad, fov_half_alpha,
                                                fov_half_beta, nx, ny, tile_rays, rank, world, _stream_ptr(stream)))
    st._back(cs)
    return st


def _host_xu8(xu8) -> np.ndarray:
    if isinstance(xu8, torch.Tensor):
        xu8 = xu8.detach().cpu().numpy()
    return np.ascontiguousarray(np.asarray(xu8, dtype=np.float64).reshape(-1, 8))


def init_explicit(a, xu8, kind=NULL, prec=F64, renormalise_ut=False, stream=None, out: State | None = None) -> State:
    """Explicit 8-vectors of null (kind = NULL) or time-like (kind = TIMELIKE) geodesics.
    xu8: HOST array (numpy or CPU torch tensor) of shape (n, 8), float64."""
    xu8 = _host_xu8(xu8)
    n = xu8.shape[0]
    st = out if out is not None else State.empty(n, prec)
    cs = st._c()
    _check(load_library().gray2_init_explicit(C.byref(cs), a, xu8.ctypes.data_as(C.c_void_p), n, int(kind),
                                              int(renormalise_ut), _stream_ptr(stream)))
    st._back(cs)
    return st


NOALLOC_MAX_GEODESICS = 65536      # GRAY2_NOALLOC_MAX_GEODESICS of include/gray2.h


def init_explicit_noalloc(a, xu8, kind=NULL, prec=F64, renormalise_ut=False, stream=None,
                          out: State | None = None) -> State:
    """gray2_init_explicit_noalloc: init_explicit for programs that must not allocate GPU memory inside the library
    (all of it promised to another allocator, a frame loop that a device-wide wait would stall, allocation locked
    after start-up; see include/gray2.h).  The library stages through a fixed 4 MiB array instead of a buffer it
    would cudaMalloc, so at most NOALLOC_MAX_GEODESICS geodesics per call (more raises Gray2Error, EINVAL), and calls
    whose GPU work can overlap (different streams) race on that array.  Pass `out` to keep the state itself out of
    torch's allocator as well.  The host array is kept alive on the returned State (``_host``) because the copy is
    only enqueued: do not modify it before the stream has been synchronised."""
    xu8 = _host_xu8(xu8)
    n = xu8.shape[0]
    st = out if out is not None else State.empty(n, prec)
    cs = st._c()
    _check(load_library().gray2_init_explicit_noalloc(C.byref(cs), a, xu8.ctypes.data_as(C.c_void_p), n, int(kind),
                                                      int(renormalise_ut), _stream_ptr(stream)))
    st._back(cs)
    st._host = xu8
    return st


def init_timelike(a, xu8, prec=F64, renormalise_ut=False, stream=None, out: State | None = None) -> State:
    """gray2_init_timelike: explicit 8-vectors of time-like geodesics (HOST array of shape (n, 8), float64)."""
    xu8 = _host_xu8(xu8)
    n = xu8.shape[0]
    st = out if out is not None else State.empty(n, prec)
    cs = st._c()
    _check(load_library().gray2_init_timelike(C.byref(cs), a, xu8.ctypes.data_as(C.c_void_p), n,
                                              int(renormalise_ut), _stream_ptr(stream)))
    st._back(cs)
    return st


def integrate(st: State, lambda_end, sc: StepControl, n=None, stats: torch.Tensor | None = None, stream=None):
    """Enqueue the integration.  `stats`: optional cuda int64 tensor of 6 entries, overwritten with
    (steps, n_captured, n_escaped, n_maxsteps, n_invalid, n_active); returned as given."""
    cs = st._c()
    sp = C.c_void_p(stats.data_ptr()) if stats is not None else C.c_void_p(0)
    if stats is not None:
        assert stats.is_cuda and stats.dtype == torch.int64 and stats.numel() >= 6
    _check(load_library().gray2_integrate(C.byref(cs), st.n if n is None else n, float(lambda_end), C.byref(sc),
                                          st.prec, sp, _stream_ptr(stream)))
    return stats


def integrate_coordtime(st: State, t_end, sc: StepControl, n=None, stats: torch.Tensor | None = None, stream=None):
    """Coordinate-time form (paper eq. 18): advance every ACTIVE geodesic to KS time t_end (see gray2.h)."""
    cs = st._c()
    sp = C.c_void_p(stats.data_ptr()) if stats is not None else C.c_void_p(0)
    if stats is not None:
        assert stats.is_cuda and stats.dtype == torch.int64 and stats.numel() >= 6
    _check(load_library().gray2_integrate_coordtime(C.byref(cs), st.n if n is None else n, float(t_end),
                                                    C.byref(sc), st.prec, sp, _stream_ptr(stream)))
    return stats


DIAG_FIELDS = ("max_abs_u2", "cos_peak", "dphi_cycle", "t_zmax1", "t_zmax2")


def integrate_diagnostics(st: State, lambda_end, sc: StepControl, n=None, stats: torch.Tensor | None = None,
                          stream=None) -> dict:
    """gray2_integrate_diagnostics: integrate and return the paper's convergence diagnostics as a dict of
    five cuda float64 tensors (see gray2_diagnostics in gray2.h)."""
    n = st.n if n is None else n
    out = torch.empty((5, n), dtype=torch.float64, device=st.q.device)
    ptrs = (C.c_void_p * 5)(*[out[k].data_ptr() for k in range(5)])
    cs = st._c()
    sp = C.c_void_p(stats.data_ptr()) if stats is not None else C.c_void_p(0)
    _check(load_library().gray2_integrate_diagnostics(C.byref(cs), n, float(lambda_end), C.byref(sc), st.prec,
                                                      C.byref(ptrs), sp, _stream_ptr(stream)))
    return dict(zip(DIAG_FIELDS, out))


def new_stats(device="cuda") -> torch.Tensor:
    return torch.zeros(6, dtype=torch.int64, device=device)


def stats_dict(stats: torch.Tensor) -> dict:
    v = stats.cpu().tolist()
    return dict(zip(STATS_FIELDS, v))


def invariants(st: State, n=None, stream=None):
    """E, Lz, Q, norm as four cuda float64 tensors (of the RUN geodesic, see gray2.h)."""
    n = st.n if n is None else n
    out = torch.empty((4, n), dtype=torch.float64, device=st.q.device)
    cs = st._c()
    _check(load_library().gray2_invariants(C.byref(cs), n, *[C.c_void_p(out[k].data_ptr()) for k in range(4)],
                                           _stream_ptr(stream)))
    return out[0], out[1], out[2], out[3]


def rhs(prec, a, pos: torch.Tensor, u: torch.Tensor, stream=None) -> torch.Tensor:
    """Diagnostic: geodesic right-hand side at n points.  pos (3, n), u (4, n) cuda tensors -> (4, n)."""
    dt = torch.float64 if prec == F64 else torch.float32
    pos = pos.to(dt).contiguous()
    u = u.to(dt).contiguous()
    n = pos.shape[1]
    out = torch.empty((4, n), dtype=dt, device=pos.device)
    _check(load_library().gray2_rhs(prec, a, n, C.c_void_p(pos.data_ptr()), C.c_void_p(u.data_ptr()),
                                    C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def rhs_bl(prec, a, pos: torch.Tensor, u: torch.Tensor, stream=None) -> torch.Tensor:
    """Diagnostic: Boyer-Lindquist right-hand side at n points.  pos (2, n) = r, theta; u (4, n) -> (4, n)."""
    dt = torch.float64 if prec == F64 else torch.float32
    pos = pos.to(dt).contiguous()
    u = u.to(dt).contiguous()
    n = pos.shape[1]
    out = torch.empty((4, n), dtype=dt, device=pos.device)
    _check(load_library().gray2_rhs_bl(prec, a, n, C.c_void_p(pos.data_ptr()), C.c_void_p(u.data_ptr()),
                                       C.c_void_p(out.data_ptr()), _stream_ptr(stream)))
    return out


def convert(st: State, to_coords: int, n=None, stream=None, out: State | None = None) -> State:
    """The same geodesics in the other coordinate system (KS <-> BL), as a new State (or into `out`)."""
    n = st.n if n is None else n
    dst = out if out is not None else State.empty(st.n, st.prec, st.q.device)
    cs, cd = st._c(), dst._c()
    _check(load_library().gray2_convert(C.byref(cs), C.byref(cd), n, to_coords, _stream_ptr(stream)))
    dst._back(cd)
    return dst


def order_longest_first(steps_hint: torch.Tensor, stream=None, out: torch.Tensor | None = None) -> torch.Tensor:
    """gray2_order_longest_first: the indices sorted by decreasing steps_hint (cuda int32), as a cuda int32 tensor
    to put into State.order."""
    assert steps_hint.is_cuda and steps_hint.dtype == torch.int32 and steps_hint.is_contiguous()
    n = steps_hint.numel()
    order = out if out is not None else torch.empty(n, dtype=torch.int32, device=steps_hint.device)
    _check(load_library().gray2_order_longest_first(C.c_void_p(steps_hint.data_ptr()), n, C.c_void_p(order.data_ptr()),
                                                    _stream_ptr(stream)))
    return order


def set_launch(prec, threads_per_block=0, blocks_per_sm=0):
    _check(load_library().gray2_set_launch(prec, threads_per_block, blocks_per_sm))


def flops_per_step(prec=F64) -> int:
    return int(load_library().gray2_flops_per_step(prec))


def flops_per_step_coordtime(prec=F64) -> int:
    return int(load_library().gray2_flops_per_step_coordtime(prec))


def flops_per_step_bl(prec=F64) -> int:
    return int(load_library().gray2_flops_per_step_bl(prec))


def version() -> str:
    return load_library().gray2_version().decode()
