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
    assert lib.gray2_flops_per_step(0) == 530 and lib.gray2_flops_per_step(1) == 554


def test_struct_layouts_match_the_header(lib):
    from paper_1706_07062_b200 import gray2
    # gray2_state: 8 pointers + 3 pointers + u64 + double + 4 int32 + the order pointer ; gray2_step_control per the header
    assert C.sizeof(gray2._CState) == 8 * 8 + 3 * 8 + 8 + 8 + 16 + 8 and gray2._CState.order.offset == 120
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


def test_new_entries_reject_bad_arguments_without_gpu_work(lib):
    from paper_1706_07062_b200 import gray2
    EINVAL, ESTATE = 1, 2
    null = C.c_void_p(0)
    assert gray2._CState.coords.offset == 116 and gray2._CState.reversed.offset == 112
    s = gray2._CState()
    s.n, s.prec = 16, 0
    for m in range(8):
        s.q[m] = 0x1000
    s.lam = s.status = s.nsteps = 0x1000
    d = gray2._CState()
    C.memmove(C.byref(d), C.byref(s), C.sizeof(s))
    assert lib.gray2_convert(C.byref(s), C.byref(d), 16, 0, null) == EINVAL          # already Kerr-Schild
    assert lib.gray2_convert(C.byref(s), C.byref(d), 16, 5, null) == EINVAL          # unknown coordinates
    assert lib.gray2_convert(C.byref(s), null, 16, 1, null) == EINVAL
    assert lib.gray2_convert(C.byref(s), C.byref(d), 17, 1, null) == ESTATE
    d.prec = 1
    assert lib.gray2_convert(C.byref(s), C.byref(d), 16, 1, null) == EINVAL          # precision mismatch
    assert d.coords == 0                                                              # dst untouched on error
    s.coords = 9
    sc = gray2.step_control(mode=1, eta=0.01)
    assert lib.gray2_integrate(C.byref(s), 16, 1.0, C.byref(sc), 0, null, null) == EINVAL
    s.coords = 1                                                                       # Boyer-Lindquist state
    assert lib.gray2_integrate_coordtime(C.byref(s), 16, 1.0, C.byref(sc), 0, null, null) == EINVAL
    s.coords = 0
    lib.gray2_init_null_shard.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double,
                                          C.c_int32, C.c_int32, C.c_uint64, C.c_int32, C.c_int32, C.c_void_p]
    args = (0.5, 100.0, 1.0, 10.0, 10.0, 8, 4)
    assert lib.gray2_init_null_shard(C.byref(s), *args, 0, 0, 2, null) == EINVAL      # tile_rays == 0
    assert lib.gray2_init_null_shard(C.byref(s), *args, 8, 2, 2, null) == EINVAL      # rank >= world
    s.n = 15
    assert lib.gray2_init_null_shard(C.byref(s), *args, 8, 0, 2, null) == EINVAL      # shard has 16 rays, state 15
    assert lib.gray2_rhs_bl(0, 0.5, 0, null, null, null, null) == EINVAL
    assert lib.gray2_flops_per_step_bl(0) == 598 and lib.gray2_flops_per_step_bl(1) == 590
    assert lib.gray2_flops_per_step_coordtime(0) == 534 and lib.gray2_flops_per_step_coordtime(1) == 574
    fake = C.c_void_p(0x1000)
    s.n = 16
    assert lib.gray2_init_explicit(C.byref(s), 0.5, fake, 16, 7, 0, null) == EINVAL   # unknown kind
    assert b"kind" in lib.gray2_last_error()
    assert lib.gray2_init_explicit(C.byref(s), 0.5, null, 16, 0, 0, null) == EINVAL   # no host array
    assert lib.gray2_init_explicit(C.byref(s), 0.5, fake, 17, 0, 0, null) == ESTATE   # n > s->n
    assert lib.gray2_init_explicit(C.byref(s), 1.5, fake, 16, 1, 0, null) == EINVAL   # |a| > 1
    assert lib.gray2_order_longest_first(null, 16, fake, null) == EINVAL              # no hint array
    assert lib.gray2_order_longest_first(fake, 0, fake, null) == EINVAL               # n == 0
    assert lib.gray2_order_longest_first(fake, 1 << 31, fake, null) == EINVAL         # indices are int32
    assert not hasattr(lib, "gray2_fma_probe")        # the probe kernels live in bench_probe.cu, not in the product


def test_bench_reference_arm_prints_the_contract_line():
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0", "--oracle-side", "16"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-500:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["vs_baseline"] is None and line["higher_is_better"] is True
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "scaling", "dtype", "data", "config"):
        assert key in line, key
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["value"] > 1e4 and line["config"]["rays"] == 256


def test_bench_gpu_arm_fails_loudly_without_a_gpu():
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "1"], capture_output=True,
                         text=True, timeout=300)
    assert out.returncode != 0 and "no CPU fallback" in (out.stderr + out.stdout)


def test_bench_gpus_n_without_the_devices_fails_loudly():
    """`bench.py --gpus 2` outside torchrun starts the ranks itself; on a box with fewer than 2 GPUs it must say so
    and exit non-zero instead of printing a one-rank line."""
    import subprocess
    import sys
    import torch
    if torch.cuda.is_available() and torch.cuda.device_count() >= 2:
        pytest.skip("two GPUs are present")
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode != 0 and "needs 2 CUDA devices" in (out.stderr + out.stdout)
    assert "n_gpus" not in out.stdout


def test_bench_probe_object_builds_and_is_separate_from_the_product():
    import subprocess
    sys_path = os.path.join(ROOT, "bench_probe.cu")
    assert os.path.exists(sys_path)
    import bench                                            # bench.py at the repo root (conftest puts it on sys.path)
    lib = C.CDLL(bench.build_probe())
    assert hasattr(lib, "bench_fma_probe")
    assert lib.bench_fma_probe(0, 3, 1, 32, 1, C.c_void_p(0x1000), None) == 1        # packed form is FP32 only
    assert lib.bench_fma_probe(1, 2, 1, 32, 1, None, None) == 1                      # no scratch
    assert bench.load_counters("cfg3", "f64", "affine") is not None


def test_bench_line_blocks_are_assembled_from_the_measurements():
    """bench.block_of (the JSON fields of one precision) from synthetic per-rank measurements: no GPU needed.
    Checks the arithmetic of value / roofline / executed_frac / e2e and that the profiler-only figures come from
    profiles/kernel_counters.csv."""
    import types
    import bench
    F64, F32 = 0, 1
    flops = {F64: 530, F32: 554}
    gray2 = types.SimpleNamespace(F64=F64, F32=F32)
    args = types.SimpleNamespace(steps=2, workload="cfg3", form="affine")
    job = types.SimpleNamespace(args=args, cfg=None, gray2=gray2, n_sms=148, sm_max_mhz=1965.0, world=1, strong=False,
                                coord=False, bl=False, n_local=1 << 20, flops_per_step=lambda prec: flops[prec])
    for dtype, prec in (("f64", F64), ("f32", F32)):
        m = dict(dtype=dtype, prec=prec, per_step=[0.030, 0.028], per_int=[0.0295, 0.0275], steps_total=2_200_000_000,
                 clocks={"sm_mhz": 1965.0, "reasons": []}, h2d=64, d2h=80, n_chunks=32, n_streams=8,
                 probe={"imm": 36.0, "regs": 34.0, "fresh": 24.6, "packed": 48.7}, warmup=3,
                 per_init=[17e-6, 19e-6], per_inv=[16e-6, 16e-6])
        b = bench.block_of(job, m, t_step=0.058, t_int=0.057, steps_all=2.2e9, t_e2e=0.06, e2e_all=2.2e9)
        peak = 148 * (64 if dtype == "f64" else 128) * 2 * 1965e6 / 1e12
        assert abs(b["value"] - 2.2e9 / 0.058) < 1 and abs(b["ms_per_step"] - 29.0) < 1e-9
        assert abs(b["ms_per_step_best"] - 28.0) < 1e-9 and abs(b["ms_per_step_median"] - 29.0) < 1e-9
        r = b["roofline"]
        assert abs(r["peak"] - peak) < 1e-9 and r["bound"] == "alu" and r["unit"] == "TFLOP/s"
        assert abs(r["achieved"] - 2.2e9 * flops[prec] / 0.057 / 1e12) < 1e-9 and abs(r["frac"] - r["achieved"] / peak) < 1e-12
        row = bench.load_counters("cfg3", dtype, "affine")
        assert r["traffic"] == int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
        assert abs(r["executed_frac"] - 2.2e9 * float(row["executed_flops_per_step"]) / 0.057 / 1e12 / peak) < 1e-12
        assert r["algorithmic_bytes"] == 2 * (80 if dtype == "f64" else 48) * (1 << 20)
        assert b["e2e"]["h2d_bytes_per_step"] == 64 and abs(b["e2e"]["value"] - 2.2e9 / 0.06) < 1
        assert b["gpu_launches"] == 8
        assert abs(b["init_ms"] - 0.018) < 1e-12 and abs(b["invariants_ms"] - 0.016) < 1e-12
        assert r["counters_match_this_build"] == (row.get("csrc_sha12") == bench.csrc_digest())
        if dtype == "f32":
            assert abs(r["frac_without_compensation_flops"] - r["frac"] * 530 / 554) < 1e-12
    assert bench.load_counters("cfg9", "f64", "affine") is None


def test_noalloc_entry_states_its_limit_and_refuses_more_without_gpu_work(lib):
    """gray2_init_explicit_noalloc stages through a fixed array (include/gray2.h): the limit is in the header, the
    binding repeats it, and a larger batch is refused before any CUDA call with an error that names it."""
    from paper_1706_07062_b200 import gray2
    text = open(os.path.join(ROOT, "include", "gray2.h")).read()
    limit = int(re.search(r"#define\s+GRAY2_NOALLOC_MAX_GEODESICS\s+(\d+)", text).group(1))
    assert limit == gray2.NOALLOC_MAX_GEODESICS and limit * 64 == 4 << 20
    s = gray2._CState()
    s.n, s.prec = 1 << 20, 0
    for m in range(8):
        s.q[m] = 0x1000
    s.lam = s.status = s.nsteps = 0x1000
    fake, null = C.c_void_p(0x1000), C.c_void_p(0)
    assert lib.gray2_init_explicit_noalloc(C.byref(s), 0.5, fake, limit + 1, 0, 0, null) == gray2.EINVAL
    assert b"GRAY2_NOALLOC_MAX_GEODESICS" in lib.gray2_last_error() and str(limit).encode() in lib.gray2_last_error()
    assert lib.gray2_init_explicit_noalloc(C.byref(s), 0.5, null, 16, 0, 0, null) == gray2.EINVAL     # no host array
    assert lib.gray2_init_explicit_noalloc(C.byref(s), 0.5, fake, 16, 7, 0, null) == gray2.EINVAL     # unknown kind
    s.n = 8
    assert lib.gray2_init_explicit_noalloc(C.byref(s), 0.5, fake, 16, 0, 0, null) == gray2.ESTATE     # n > s->n
