"""gray2_init_explicit_noalloc against gray2_init_explicit (GPU).

Some programs that call this library cannot let it allocate GPU memory: they have promised (nearly) all of it to
an allocator of their own, or they run a frame loop that the device-wide wait inside cudaMalloc / cudaFree would
stall, or they lock allocation down once they have started.  gray2_init_explicit is the one call that may allocate
at any time (it regrows its staging buffer whenever a batch is larger than before), so it has a twin that stages
through a fixed 4 MiB array inside the library instead (include/gray2.h).  Same kernel, so the test asks for the
same state BIT FOR BIT -- tighter than the 1e-14 the init tests grant against the oracle -- on two calls in a row:
the second call finds the array full of the first call's geodesics and must not see any of them.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should not hide the
parity tests.  Nothing here depends on what ran before (it passes alone in a fresh process and after the others)."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_1706_07062_b200 import gray2, inputs

pytestmark = pytest.mark.gpu


def _same_state(got: gray2.State, want: gray2.State, n: int):
    torch.cuda.synchronize()
    assert (got.a_eff, got.kind, got.reversed, got.coords) == (want.a_eff, want.kind, want.reversed, want.coords)
    # bit patterns, so that a NaN or a signed zero cannot hide a difference
    bits = torch.int64 if got.q.dtype == torch.float64 else torch.int32
    assert torch.equal(got.q[:, :n].contiguous().view(bits), want.q[:, :n].contiguous().view(bits))
    assert torch.equal(got.lam[:n], want.lam[:n])
    assert torch.equal(got.status[:n], want.status[:n]) and torch.equal(got.nsteps[:n], want.nsteps[:n])


def test_two_calls_in_a_row_equal_the_allocating_path():
    # call 1: 5,003 bound particles (20 blocks, the last one ragged), double, u^t solved on the device
    xu8, _ = inputs.cfg4_ensemble(5003)
    first = xu8.copy()
    first[:, 4] = 99.0                                  # replaced by the root of g u u = -1
    want = gray2.init_explicit(0.7, first, gray2.TIMELIKE, renormalise_ut=True)
    got = gray2.init_explicit_noalloc(0.7, first, gray2.TIMELIKE, renormalise_ut=True)
    _same_state(got, want, 5003)

    # call 2, straight after it on the same stream: fewer geodesics, other numbers, photons, float.  The array
    # still holds call 1's particles from row 1,237 on; the state must show none of them.
    rng = np.random.default_rng(1706)
    second = rng.uniform(-30.0, 30.0, (1237, 8))
    second[:, 4] = rng.uniform(1.0, 3.0, 1237)
    want2 = gray2.init_explicit(-0.9375, second, gray2.NULL, prec=gray2.F32)
    got2 = gray2.init_explicit_noalloc(-0.9375, second, gray2.NULL, prec=gray2.F32)
    _same_state(got2, want2, 1237)
    assert got2.q.dtype == torch.float32 and got2.kind == gray2.NULL

    # and the states the new entry makes are ordinary states: the integrator takes them like any other
    sc = gray2.step_control(mode=0, h_fixed=0.5, max_steps=40)
    gray2.integrate(got, float("inf"), sc)
    gray2.integrate(want, float("inf"), sc)
    _same_state(got, want, 5003)
    assert int(got.nsteps.max()) == 40


def test_a_full_array_and_one_geodesic_too_many():
    n = gray2.NOALLOC_MAX_GEODESICS
    rng = np.random.default_rng(62)
    xu8 = rng.uniform(-50.0, 50.0, (n + 1, 8))
    xu8[:, 4] = rng.uniform(1.0, 2.0, n + 1)
    # exactly the maximum: every byte of the array is used, the last row included
    want = gray2.init_explicit(0.5, xu8[:n], gray2.NULL)
    got = gray2.init_explicit_noalloc(0.5, xu8[:n], gray2.NULL)
    _same_state(got, want, n)
    # one more is refused with an error that names the limit, and nothing has been written
    out = gray2.State.empty(n + 1)
    out.q.fill_(-7.0)
    with pytest.raises(gray2.Gray2Error) as err:
        gray2.init_explicit_noalloc(0.5, xu8, gray2.NULL, out=out)
    assert err.value.code == gray2.EINVAL
    assert str(n) in str(err.value) and "GRAY2_NOALLOC_MAX_GEODESICS" in str(err.value)
    torch.cuda.synchronize()
    assert bool((out.q == -7.0).all())
    # the limit in the header is the one the binding states
    lib = gray2.load_library()
    s = out._c()
    assert lib.gray2_init_explicit_noalloc(C.byref(s), 0.5, xu8.ctypes.data_as(C.c_void_p), n + 1, 0, 0, None) == gray2.EINVAL
