"""The C-ABI library: it loads without a GPU, exports every function include/gray2.h declares, and
rejects bad arguments before doing any GPU work.  CPU only (no compute call is made)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1706_07062_b200 import build
    build.build()
    from paper_1706_07062_b200 import gray2
    return gray2.load_library()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gray2.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gray2_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_four_calls():
    names = declared_functions()
    for required in ("gray2_init_null", "gray2_init_timelike", "gray2_integrate", "gray2_invariants"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.gray2_version()
    assert lib.gray2_flops_per_step(0) == 530 and lib.gray2_flops_per_step(1) == 530


def test_struct_layouts_match_the_header(lib):
    from paper_1706_07062_b200 import gray2
    # gray2_state: 8 pointers + 3 pointers + u64 + double + 3 int32 (+ pad) ; gray2_step_control per the header
    assert C.sizeof(gray2._CState) == 8 * 8 + 3 * 8 + 8 + 8 + 16
    assert C.sizeof(gray2.StepControl) == 56
    assert gray2.StepControl.eta.offset == 16 and gray2.StepControl.max_steps.offset == 48


def test_bad_arguments_are_rejected_without_gpu_work(lib):
    from paper_1706_07062_b200 import gray2
    EINVAL, ESTATE = 1, 2
    null = C.c_void_p(0)
    assert lib.gray2_init_null(null, 0.5, 100.0, 1.0, 10.0, 10.0, 4, 4, null) == EINVAL
    assert b"NULL" in lib.gray2_last_error()
    s = gray2._CState()
    s.n = 16
    s.prec = 0
    assert lib.gray2_init_null(C.byref(s), 0.5, 100.0, 1.0, 10.0, 10.0, 4, 4, null) == EINVAL  # q[] NULL
    for m in range(8):
        s.q[m] = 0x1000
    s.lam = s.status = s.nsteps = 0x1000
    assert lib.gray2_init_null(C.byref(s), 1.5, 100.0, 1.0, 10.0, 10.0, 4, 4, null) == EINVAL   # |a| > 1
    assert lib.gray2_init_null(C.byref(s), 0.5, 100.0, 1.0, 10.0, 10.0, 4, 5, null) == EINVAL   # nx*ny != n
    assert lib.gray2_init_null(C.byref(s), 0.5, 1.2, 1.0, 10.0, 10.0, 4, 4, null) == EINVAL     # r_obs <= r_plus
    sc = gray2.step_control(mode=1, eta=0.0)
    assert lib.gray2_integrate(C.byref(s), 16, 1.0, C.byref(sc), 0, null, null) == EINVAL       # eta <= 0
    sc = gray2.step_control(mode=1, eta=0.01)
    assert lib.gray2_integrate(C.byref(s), 16, 1.0, C.byref(sc), 1, null, null) == EINVAL       # prec mismatch
    assert lib.gray2_integrate(C.byref(s), 0, 1.0, C.byref(sc), 0, null, null) == EINVAL        # n == 0
    assert lib.gray2_integrate(C.byref(s), 17, 1.0, C.byref(sc), 0, null, null) == ESTATE       # n > s->n
    sc = gray2.step_control(mode=1, eta=0.01, dir=0)
    assert lib.gray2_integrate(C.byref(s), 16, 1.0, C.byref(sc), 0, null, null) == EINVAL       # dir
    assert lib.gray2_integrate(C.byref(s), 16, 1.0, null, 0, null, null) == EINVAL              # sc NULL
    assert lib.gray2_invariants(C.byref(s), 16, null, null, null, null, null) == EINVAL
    assert lib.gray2_init_timelike(C.byref(s), 0.5, null, 16, 0, null) == EINVAL
    assert lib.gray2_set_launch(0, 96, 5) == EINVAL and lib.gray2_set_launch(0, 0, 0) == 0
    assert lib.gray2_rhs(0, 0.5, 0, null, null, null, null) == EINVAL


def test_binding_refuses_to_run_without_a_gpu():
    import torch
    from paper_1706_07062_b200 import gray2
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        gray2.init_null(0.5, 100.0, 1.0, 10.0, 10.0, 4, 4)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1706_07062_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "gray2_oracle" not in text, f
