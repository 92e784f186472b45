#!/usr/bin/env python
"""bench.py -- geodesic RK4 steps/s of the whole hot path on BASELINE.json's headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype both|f64|f32] [--workload cfg3|cfg1|cfg2|cfg5]
    python bench.py --impl reference ...      # the oracle, as it stands, on the host cores

A "step" is one pass of the whole path over one batch: gray2_init_null (image-plane initial conditions)
-> gray2_integrate (fused RHS + RK4 + termination + refill) -> gray2_invariants, on the 1024 x 1024
Kerr image of BASELINE.json configs[2] ("cfg3": a = 0.9375, r_obs = 1000 M, i = 60 deg, +-15 M), which is
the workload north_star quotes the target on.  The metric is geodesic RK4 steps per second (whole job,
summed over ranks; each rank traces its own image: weak scaling, no collective on the data path;
--scaling strong shares ONE image among the ranks in tiles of 4096 rays, again without a collective).

BASELINE.json's metric names both precisions, so the default run (--dtype both) times FP64 and then FP32 on
the same workload: the top-level fields of the JSON line are the FP64 run (BASELINE dtype), the block
"fp32" carries the same fields for the FP32 run, and "both" the two integrations enqueued together on two
streams against their serial sum (cfg3 is specified "in both FP64 and FP32").

--gpus N: under torchrun (WORLD_SIZE set) this process is one of the N ranks; without it bench.py starts the
N ranks itself, one process per GPU, and fails if the box has fewer than N devices.

One JSON line is printed by rank 0; see DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import csv
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "geodesic RK4 steps/sec on 1 B200 (FP64, FP32) and fraction of non-tensor FP peak"
UNIT = "RK4 steps/s"
SHARD_TILE = 4096          # rays per tile when one image is shared by several GPUs (--scaling strong)
INF = float("inf")

# Non-tensor FP peak of a B200 from unit counts and clocks: 148 SMs x 64 FP64 lanes
# (128 FP32 lanes) x 2 flops per FMA x 1.965 GHz (clocks.max.sm of this pool, MEASURED_PEAKS.json).
FP_LANES = {"f64": 64, "f32": 128}

# Counters of the dominant kernel that only a profiler can give (DRAM bytes per launch from `ncu --set full`,
# executed FP thread instructions per RK4 step from the ncu op counters / the SASS of the loop) are read from
# the tracked summary below, keyed by workload, dtype and form; the commands that produced each row are in the
# .md beside it.  A workload that has no row reports null.
COUNTERS_CSV = os.path.join(ROOT, "profiles", "kernel_counters.csv")

PROBE_SRC = os.path.join(ROOT, "bench_probe.cu")
PROBE_LIB = os.path.join(ROOT, "libbench_probe.so")


def nominal_peak_tflops(dtype: str, n_sms: int, sm_max_mhz: float) -> float:
    return n_sms * FP_LANES[dtype] * 2.0 * sm_max_mhz * 1e6 / 1e12


def load_measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


def csrc_digest() -> str:
    """First 12 hex digits of the SHA-256 over the library's kernel sources and its header (sorted by name): the
    stamp of profiles/kernel_counters.csv rows (column csrc_sha12), so that a row captured on other kernels shows."""
    import hashlib
    csrc = os.path.join(ROOT, "paper_1706_07062_b200", "csrc")
    h = hashlib.sha256()
    for path in sorted(os.path.join(csrc, f) for f in os.listdir(csrc)) + [os.path.join(ROOT, "include", "gray2.h")]:
        with open(path, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def load_counters(workload: str, dtype: str, form: str):
    """Row of profiles/kernel_counters.csv for (workload, dtype, form), or None."""
    try:
        with open(COUNTERS_CSV) as fh:
            for row in csv.DictReader(r for r in fh if not r.startswith("#")):
                if (row["workload"], row["dtype"], row["form"]) == (workload, dtype, form):
                    return row
    except Exception:
        pass
    return None


def build_probe(force: bool = False) -> str:
    """Compile bench_probe.cu (FMA-only probe kernels; bench-side, not part of libgray2.so) for sm_100a."""
    if force or not os.path.exists(PROBE_LIB) or os.path.getmtime(PROBE_LIB) < os.path.getmtime(PROBE_SRC):
        tmp = PROBE_LIB + ".tmp.%d" % os.getpid()
        nvcc = next((c for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc") if c and os.path.exists(c)), "nvcc")
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                               "--shared", "-Xcompiler", "-fPIC", "--fmad=false", "-I", ROOT, "-o", tmp, PROBE_SRC])
        os.replace(tmp, PROBE_LIB)
    return PROBE_LIB


def load_probe():
    import ctypes as C
    lib = C.CDLL(build_probe())
    lib.bench_fma_probe.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
    lib.bench_fma_probe.restype = C.c_int
    return lib


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons (profiling recipe).  It is started before the warm-up
    so that nvidia-smi's start-up cost is not inside the timed region; every sample is stamped on arrival
    and only the samples that fall inside a timed window are reported."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.samples = []          # (arrival time, fields)
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.samples.append((time.perf_counter(), line.strip()))

    def wait_for_first_sample(self, timeout=3.0):
        t0 = time.perf_counter()
        while self.proc is not None and not self.samples and time.perf_counter() - t0 < timeout:
            time.sleep(0.01)

    def window(self, t_begin, t_end) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        sm, smax, power, reasons = [], [], [], set()
        for stamp, ln in list(self.samples):
            if not (t_begin <= stamp <= t_end + 0.03):
                continue
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(self.NAMES, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples inside the timed window"]}
        return {"sm_mhz": statistics.median(sm), "sm_min_mhz": min(sm), "sm_max_mhz": max(smax),
                "power_w_max": max(power), "samples": len(sm), "reasons": sorted(reasons)}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


def workload_config(name: str):
    from paper_1706_07062_b200 import inputs
    return {"cfg1": inputs.CFG1_NULL, "cfg2": inputs.CFG2_NULL, "cfg3": inputs.CFG3_NULL,
            "cfg5": inputs.CFG5_NULL}[name]


# ---------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on the host cores, on a bounded sample
# ---------------------------------------------------------------------------------------------------

def time_oracle(cfg, side: int, steps: int, warmup: int):
    """Each step = init_null + integrate + invariants of the workload's field of view sampled on side^2 rays."""
    import oracle
    sub = cfg.scaled(side)
    sc = oracle.step_control(mode=1, eta=sub.eta, r_escape=sub.r_escape, max_steps=sub.max_steps,
                             capture_factor=sub.capture_factor)
    total_steps, total_t = 0, 0.0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        st = oracle.init_null(sub.a, sub.r_obs, sub.inclination, sub.fov, sub.fov, sub.nx, sub.ny)
        stats = oracle.integrate(st, INF, sc)
        oracle.invariants(st)
        dt = time.perf_counter() - t0
        if it >= warmup:
            total_steps += stats["steps"]
            total_t += dt
    return total_steps / total_t, total_t / steps, oracle.num_threads(), sub


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = workload_config(args.workload)
    side = args.oracle_side
    value, s_per_step, cores, sub = time_oracle(cfg, side, max(args.steps, 1), args.warmup)
    sample = "%s field of view on %dx%d rays (every %dth pixel row/column), oracle init+integrate+invariants" % (
        args.workload, side, side, cfg.nx // side)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * s_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": sub.name, "rays": sub.n, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------

class Job:
    """What every measurement of one rank shares: the workload, the device, the rank layout."""

    def __init__(self, args):
        import torch
        import torch.distributed as dist
        from paper_1706_07062_b200 import gray2
        self.args, self.torch, self.dist, self.gray2 = args, torch, dist, gray2
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        if self.world != args.gpus:
            raise SystemExit("bench.py: --gpus %d but WORLD_SIZE = %d" % (args.gpus, self.world))
        if torch.cuda.device_count() <= self.local:
            raise SystemExit("bench.py: rank %d needs cuda:%d but the box has %d device(s)"
                             % (self.rank, self.local, torch.cuda.device_count()))
        torch.cuda.set_device(self.local)
        if self.world > 1:
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
        if self.rank == 0:                       # in-tree builds (no-ops when the libraries are up to date)
            from paper_1706_07062_b200 import build as _build
            _build.build()
            build_probe()
        if self.world > 1:
            dist.barrier()
        gray2.load_library()
        self.probe_lib = load_probe()
        self.cfg = workload_config(args.workload)
        self.props = torch.cuda.get_device_properties(self.local)
        self.n_sms = self.props.multi_processor_count
        self.sm_max_mhz = float(load_measured_peaks().get("sm_max_mhz", 1965.0))
        self.coord = args.form == "coordtime"
        self.bl = args.form == "bl"     # Boyer-Lindquist variant (Table 2 "BL" rows): init -> convert -> integrate
        cfg = self.cfg
        self.sc = gray2.step_control(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                                     capture_factor=cfg.capture_factor)
        # --scaling strong: ONE image shared by all ranks, rays dealt out in tiles of 4096;
        # weak (default): every rank traces its own image.  Neither has a collective on the data path.
        self.strong = args.scaling == "strong" and self.world > 1
        self.n_local = gray2.shard_count(cfg.n, SHARD_TILE, self.rank, self.world) if self.strong else cfg.n
        self.flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        try:
            uuid = str(self.props.uuid)
            gpu_id = uuid if uuid.startswith("GPU-") else "GPU-" + uuid
        except Exception:
            gpu_id = str(self.local)
        self.sampler = ClockSampler(gpu_id)
        self.sampler.start()

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def prec_of(self, dtype):
        return self.gray2.F64 if dtype == "f64" else self.gray2.F32

    def init_image(self, prec, out=None, stream=None):
        g, cfg = self.gray2, self.cfg
        if self.strong:
            return g.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, SHARD_TILE,
                                     self.rank, self.world, prec=prec, out=out, stream=stream)
        return g.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec, out=out,
                           stream=stream)

    def flops_per_step(self, prec):
        g = self.gray2
        return (g.flops_per_step_coordtime(prec) if self.coord else g.flops_per_step_bl(prec) if self.bl
                else g.flops_per_step(prec))

    def integrate(self, *a, **kw):
        return (self.gray2.integrate_coordtime if self.coord else self.gray2.integrate)(*a, **kw)


def measure(job: Job, dtype: str) -> dict:
    """Device-resident timing, end-to-end timing and pipe probes of one precision on this rank.  Returns raw
    per-rank numbers (times in seconds, work in RK4 steps); run_gpu reduces them over the ranks."""
    torch, gray2, args, cfg = job.torch, job.gray2, job.args, job.cfg
    prec = job.prec_of(dtype)
    if args.threads or args.blocks:
        gray2.set_launch(prec, args.threads, args.blocks)
    n_local, bl = job.n_local, job.bl
    st = gray2.State.empty(n_local, prec)
    st_ks = gray2.State.empty(n_local, prec) if bl else st
    stats = gray2.new_stats()
    stream = torch.cuda.current_stream()

    def one_step(ev=None):
        if ev: ev[0].record(stream)
        job.init_image(prec, out=st_ks)
        if bl: gray2.convert(st_ks, gray2.BL, out=st)
        if ev: ev[1].record(stream)
        job.integrate(st, INF, job.sc, stats=stats)
        if ev: ev[2].record(stream)
        inv = gray2.invariants(st)
        if ev: ev[3].record(stream)
        return inv

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        one_step()
    torch.cuda.synchronize()
    job.sampler.wait_for_first_sample()

    # ---- device-resident: exactly K steps, L2 flushed before each, CUDA events on the launching stream
    job.barrier()
    t_window0 = time.perf_counter()
    per_step, per_int, per_init, per_inv, steps_total = [], [], [], [], 0
    for _ in range(args.steps):
        job.flush.fill_(1)                                     # flush L2 between timed iterations (untimed)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        one_step(ev)
        ev[3].synchronize()
        per_step.append(ev[0].elapsed_time(ev[3]) * 1e-3)
        per_int.append(ev[1].elapsed_time(ev[2]) * 1e-3)
        per_init.append(ev[0].elapsed_time(ev[1]) * 1e-3)
        per_inv.append(ev[2].elapsed_time(ev[3]) * 1e-3)
        steps_total += int(stats[0].item())
    job.barrier()
    clocks = job.sampler.window(t_window0, time.perf_counter())

    # ---- end to end through the public API with HOST buffers (pinned): H2D of the 8-vectors, D2H of results
    host_in = torch.empty((n_local, 8), dtype=torch.float64).pin_memory()
    src = job.init_image(gray2.F64)
    host_in.copy_(src.q.t())          # outside the timed region: the user's 8-vectors, resident in host memory
    a_eff = src.a_eff
    del src
    # The batch is cut into chunks that alternate between a few streams, so that the H2D copy of one chunk
    # and the D2H copy of another overlap the integration of a third (every call below is the public API).
    # Each chunk has its own contiguous device state and pinned host result buffers, so every copy is a
    # plain asynchronous memcpy.
    n_chunks = max(1, args.e2e_chunks)
    bounds = [(n_local * c // n_chunks, n_local * (c + 1) // n_chunks) for c in range(n_chunks)]
    n_streams = max(1, args.e2e_streams)
    streams = [torch.cuda.Stream() for _ in range(n_streams)]
    host_in_np = host_in.numpy()
    parts, parts_ks, host_out, chunk_stats = [], [], [], []
    for lo, hi in bounds:
        m = hi - lo
        parts.append(gray2.State.empty(m, prec))
        if bl: parts_ks.append(gray2.State.empty(m, prec))
        chunk_stats.append(gray2.new_stats())
        host_out.append(dict(q=torch.empty((8, m), dtype=st.q.dtype).pin_memory(),
                             lam=torch.empty(m, dtype=torch.float64).pin_memory(),
                             status=torch.empty(m, dtype=torch.int32).pin_memory(),
                             nsteps=torch.empty(m, dtype=torch.int32).pin_memory(),
                             inv=torch.empty((4, m), dtype=torch.float64).pin_memory(),
                             stats=torch.empty(6, dtype=torch.int64).pin_memory()))
    h2d = host_in.numel() * 8
    d2h = sum(t.numel() * t.element_size() for ho in host_out for t in ho.values())

    def e2e_step():
        for c, (lo, hi) in enumerate(bounds):
            part, ho = parts[c], host_out[c]
            with torch.cuda.stream(streams[c % n_streams]):
                # explicit null 8-vectors, H2D inside the call
                if bl:
                    gray2.init_explicit(a_eff, host_in_np[lo:hi], gray2.NULL, prec=prec, out=parts_ks[c])
                    gray2.convert(parts_ks[c], gray2.BL, out=part)
                else:
                    gray2.init_explicit(a_eff, host_in_np[lo:hi], gray2.NULL, prec=prec, out=part)
                job.integrate(part, INF, job.sc, stats=chunk_stats[c])
                inv = gray2.invariants(part)
                ho["q"].copy_(part.q, non_blocking=True); ho["lam"].copy_(part.lam, non_blocking=True)
                ho["status"].copy_(part.status, non_blocking=True); ho["nsteps"].copy_(part.nsteps, non_blocking=True)
                for k in range(4):
                    ho["inv"][k].copy_(inv[k], non_blocking=True)
                ho["stats"].copy_(chunk_stats[c], non_blocking=True)
        torch.cuda.synchronize()
        return sum(int(ho["stats"][0]) for ho in host_out)

    e2e_step()
    e2e_n = max(1, min(args.steps, 3))
    job.barrier()
    t0 = time.perf_counter()
    e2e_steps = sum(e2e_step() for _ in range(e2e_n))
    t_e2e = time.perf_counter() - t0
    del parts, parts_ks, host_out, host_in

    # ---- FMA-only probes of the pipe at the clocks of the moment (context for the nominal peak); bench-side kernels
    scratch = torch.zeros(8, dtype=torch.float64 if prec == gray2.F64 else torch.float32, device="cuda")
    iters = 20000 if prec == gray2.F64 else 40000
    blocks, threads = job.n_sms * 8, 256
    probe = {}
    for name, regs in (("imm", 0), ("regs", 1), ("fresh", 2)) + ((("packed", 3),) if prec == gray2.F32 else ()):
        def launch():
            rc = job.probe_lib.bench_fma_probe(int(prec), regs, blocks, threads, iters, scratch.data_ptr(),
                                               stream.cuda_stream)
            if rc:
                raise RuntimeError("bench_fma_probe failed")
        launch()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        launch()
        e1.record(stream)
        e1.synchronize()
        probe[name] = (32 if regs == 3 else 16) * iters * blocks * threads / (e0.elapsed_time(e1) * 1e-3) / 1e12
    if args.threads or args.blocks:
        gray2.set_launch(prec, 0, 0)
    return dict(dtype=dtype, prec=prec, per_step=per_step, per_int=per_int, per_init=per_init, per_inv=per_inv,
                steps_total=steps_total, clocks=clocks,
                t_e2e=t_e2e, e2e_steps=e2e_steps, h2d=h2d, d2h=d2h, n_chunks=n_chunks, n_streams=n_streams,
                probe=probe, warmup=warmup)


def measure_both(job: Job) -> dict:
    """cfg3 is specified "in both FP64 and FP32 with identical step rules": the two integrations enqueued together
    on two streams (launch shapes that fit one SM's register file side by side) against the same two enqueued one
    after the other.  The FP64 kernel leaves the FP32 pipe idle and the reverse; whether they overlap is measured."""
    torch, gray2, args = job.torch, job.gray2, job.args
    s64, s32 = gray2.State.empty(job.n_local, gray2.F64), gray2.State.empty(job.n_local, gray2.F32)
    st64, st32 = gray2.new_stats(), gray2.new_stats()
    a, b = torch.cuda.Stream(), torch.cuda.Stream()

    def run(concurrent: bool):
        job.init_image(gray2.F64, out=s64)
        job.init_image(gray2.F32, out=s32)
        job.flush.fill_(1)
        torch.cuda.synchronize()
        e0, e1, eb = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(a)
        b.wait_event(e0)
        job.integrate(s64, INF, job.sc, stats=st64, stream=a)
        if not concurrent:
            mid = torch.cuda.Event()
            mid.record(a)
            b.wait_event(mid)
        job.integrate(s32, INF, job.sc, stats=st32, stream=b)
        eb.record(b)
        a.wait_event(eb)
        e1.record(a)
        e1.synchronize()
        return e0.elapsed_time(e1) * 1e-3, int(st64[0].item()) + int(st32[0].item())

    def run_fp32_first():
        """FP32 first; its step counts (equal to FP64's on 99.98 % of the rays) schedule the FP64 pass longest first
        (gray2_order_longest_first -> gray2_state.order): everything inside the timed region, outputs unchanged."""
        job.init_image(gray2.F64, out=s64)
        job.init_image(gray2.F32, out=s32)
        s64.order = None
        job.flush.fill_(1)
        torch.cuda.synchronize()
        e0, e1 = (torch.cuda.Event(enable_timing=True) for _ in range(2))
        e0.record(a)
        job.integrate(s32, INF, job.sc, stats=st32, stream=a)
        s64.order = gray2.order_longest_first(s32.nsteps, stream=a, out=order)
        job.integrate(s64, INF, job.sc, stats=st64, stream=a)
        e1.record(a)
        e1.synchronize()
        s64.order = None
        return e0.elapsed_time(e1) * 1e-3, int(st64[0].item()) + int(st32[0].item())

    order = torch.empty(job.n_local, dtype=torch.int32, device="cuda")
    out = {}
    for name, conc, shapes in (("serial", False, ((0, 0), (0, 0))), ("concurrent", True, ((128, 2), (256, 1))),
                               ("fp32_first", None, ((0, 0), (0, 0)))):
        gray2.set_launch(gray2.F64, *shapes[0])
        gray2.set_launch(gray2.F32, *shapes[1])
        fn = run_fp32_first if conc is None else (lambda: run(conc))
        for _ in range(2):
            fn()
        job.barrier()
        res = [fn() for _ in range(max(3, args.steps))]
        out[name] = dict(times=[r[0] for r in res], steps=res[0][1])
    gray2.set_launch(gray2.F64, 0, 0)
    gray2.set_launch(gray2.F32, 0, 0)
    return out


def block_of(job: Job, m: dict, t_step, t_int, steps_all, t_e2e, e2e_all) -> dict:
    """The JSON fields of one precision from its reduced numbers (rank 0)."""
    args, cfg = job.args, job.cfg
    dtype, prec = m["dtype"], m["prec"]
    fps = job.flops_per_step(prec)
    peak = nominal_peak_tflops(dtype, job.n_sms, job.sm_max_mhz)
    achieved = (m["steps_total"] * fps / sum(m["per_int"])) / 1e12            # this rank's dominant kernel
    steps_per_pass = m["steps_total"] // args.steps
    best_int = min(m["per_int"])
    row = load_counters(args.workload, dtype, args.form) or {}
    traffic = int(row["dram_read_bytes"]) + int(row["dram_write_bytes"]) if row.get("dram_read_bytes") else None
    exec_flops = float(row["executed_flops_per_step"]) if row.get("executed_flops_per_step") else None
    kernel = ("integrate_kernel<double%s>" if dtype == "f64" else "integrate_kernel_f32x2<%s>") % (
        ", coordinate time" if job.coord else ", Boyer-Lindquist" if job.bl else ("" if dtype == "f64" else "affine"))
    return {
        "value": steps_all / t_step, "unit": UNIT, "dtype": dtype,
        "ms_per_step": 1e3 * t_step / args.steps,
        "ms_per_step_best": 1e3 * min(m["per_step"]), "ms_per_step_median": 1e3 * statistics.median(m["per_step"]),
        "value_best": steps_per_pass / min(m["per_step"]) * (job.world if not job.strong else 1),
        "clocks": m["clocks"],
        "e2e": {"value": e2e_all / t_e2e, "unit": UNIT, "h2d_bytes_per_step": m["h2d"], "d2h_bytes_per_step": m["d2h"],
                "api": "gray2_init_explicit(host 8-vectors, NULL) -> %sgray2_integrate -> gray2_invariants -> D2H of state, invariants, stats"
                       % ("gray2_convert -> " if job.bl else ""),
                "chunks": m["n_chunks"], "streams": m["n_streams"]},
        # SURVEY 8(d) "also report init time, invariants time": this rank's mean per step, CUDA events around
        # gray2_init_null (+ gray2_convert for --form bl) and around gray2_invariants
        "init_ms": 1e3 * statistics.mean(m["per_init"]) if m.get("per_init") else None,
        "invariants_ms": 1e3 * statistics.mean(m["per_inv"]) if m.get("per_inv") else None,
        # kernels of this library per step: init_null, integrate, count_status, invariants (+ ks_to_bl).  gray2_integrate
        # also enqueues two memsets and one 8-byte device-to-device copy, which are not kernels of the library.
        "gpu_launches": (5 if job.bl else 4) * args.steps,
        "roofline": {"bound": "alu", "kernel": kernel,
                     "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                     "frac_best": steps_per_pass * fps / best_int / 1e12 / peak,
                     "executed_frac": (m["steps_total"] * exec_flops / sum(m["per_int"]) / 1e12 / peak) if exec_flops else None,
                     "executed_flops_per_rk4_step": exec_flops,
                     "executed_source": row.get("executed_source"),
                     # the profiler-only figures were captured on the build whose kernel sources hash to the row's
                     # csrc_sha12; False = the kernels have changed since, executed_frac and traffic describe an older build
                     "counters_match_this_build": (row.get("csrc_sha12") == csrc_digest()) if row else None,
                     "traffic": traffic,
                     "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, profiles/kernel_counters.csv)",
                     "algorithmic_bytes": 2 * (80 if dtype == "f64" else 48) * job.n_local,
                     "flops_per_rk4_step": fps,
                     # FP32 only: the same fraction with the count of the uncompensated step (round 1's: 530 affine,
                     # 534 coordinate time, 566 Boyer-Lindquist), i.e. without the 3 additions per state variable
                     "frac_without_compensation_flops": (achieved / peak) * (566 if job.bl else job.flops_per_step(job.gray2.F64)) / fps
                                                        if dtype == "f32" else None,
                     "kernel_ms": 1e3 * t_int / args.steps, "kernel_ms_best": 1e3 * best_int,
                     "kernel_share_of_step": t_int / t_step,
                     "peak_source": "nominal: %d SMs x %d lanes x 2 x %.0f MHz" % (job.n_sms, FP_LANES[dtype], job.sm_max_mhz),
                     "fma_probe_tflops": m["probe"]["imm"], "frac_of_fma_probe": achieved / m["probe"]["imm"],
                     "fma_probe_register_operands_tflops": m["probe"]["regs"],
                     "fma_probe_fresh_register_operands_tflops": m["probe"]["fresh"],
                     "fma_probe_packed_fp32x2_tflops": m["probe"].get("packed")},
    }


def run_gpu(args):
    job = Job(args)
    torch, cfg = job.torch, job.cfg
    from paper_1706_07062_b200 import multi
    dtypes = ["f64", "f32"] if args.dtype == "both" else [args.dtype]
    blocks = {}
    for dtype in dtypes:
        m = measure(job, dtype)
        # ---- reduce over ranks: time = max, work = sum
        (t_step, t_int, t_e2e), (steps_all, e2e_all) = multi.reduce_job(
            [sum(m["per_step"]), sum(m["per_int"]), m["t_e2e"]], [m["steps_total"], m["e2e_steps"]], device="cuda")
        if job.rank == 0:
            blocks[dtype] = block_of(job, m, t_step, t_int, steps_all, t_e2e, e2e_all)
            blocks[dtype]["rk4_steps_per_pass"] = m["steps_total"] // args.steps
            blocks[dtype]["warmup"] = m["warmup"]
    both = None
    if args.dtype == "both" and not job.bl and not job.coord and not args.no_both:
        b = measure_both(job)
        (ts, tc, tf), (work,) = multi.reduce_job([statistics.median(b[k]["times"]) for k in ("serial", "concurrent", "fp32_first")],
                                                 [b["serial"]["steps"]], device="cuda")
        both = {"what": "gray2_integrate FP64 and FP32 of the same image: enqueued one after the other (serial); together on "
                        "two streams with launch shapes 128x2 (FP64) + 256x1 (FP32) per SM (concurrent); FP32 first and the "
                        "FP64 pass scheduled longest first from the FP32 step counts, sort included (fp32_first_ordered)",
                "ms_serial_sum": 1e3 * ts, "ms_concurrent": 1e3 * tc, "gain": ts / tc,
                "ms_fp32_first_ordered": 1e3 * tf, "gain_fp32_first_ordered": ts / tf,
                "rk4_steps_both": int(work), "value_concurrent": work / tc, "value_fp32_first_ordered": work / tf, "unit": UNIT}
    job.sampler.stop()

    if job.rank == 0:
        head = blocks[dtypes[0]]
        line = {
            "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": job.world, "steps": args.steps,
            "warmup": head.pop("warmup"), "ms_per_step": head["ms_per_step"], "higher_is_better": True,
            "scaling": "strong" if job.strong else "weak", "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic",
            "config": {"workload": cfg.name, "rays_per_gpu": job.n_local, "rk4_steps_per_pass": head.pop("rk4_steps_per_pass"),
                       "a": cfg.a, "r_obs": cfg.r_obs, "inclination_deg": cfg.inclination_deg, "fov_half": cfg.fov,
                       "form": args.form, "step_rule": ("dt = %g r" if job.coord else "dlambda = %g r") % cfg.eta,
                       "l2": "flushed between timed iterations (256 MiB fill)",
                       "parallelism": ("one image dealt out in tiles of %d rays, no collective" % SHARD_TILE) if job.strong
                                      else "independent image per GPU, no collective"},
        }
        for k, v in head.items():
            line.setdefault(k, v)
        if len(dtypes) > 1:
            f32 = blocks["f32"]
            f32.pop("warmup", None)
            line["fp32"] = f32
        if both is not None:
            line["both"] = both
        if not args.no_cpu_baseline and job.world == 1:
            # a first pass on oracle_side^2 rays sizes the sample: about 12 s of wall clock on this box's cores
            _, s_probe, _, _ = time_oracle(cfg, args.oracle_side, 1, 0)
            side = int(args.oracle_side * math.sqrt(max(1.0, 12.0 / max(s_probe, 1e-3)))) // 32 * 32
            side = max(args.oracle_side, min(side, 512, cfg.nx))
            v, s_per, cores, sub = time_oracle(cfg, side, 1, 0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": "%s field of view on %dx%d rays, one pass (%.1f s)" % (
                                        args.workload, side, side, s_per)}
        print(json.dumps(line), flush=True)
    if job.world > 1:
        job.dist.destroy_process_group()
    return 0


# ---------------------------------------------------------------------------------------------------
# --gpus N without torchrun: start the N ranks here, one process per GPU
# ---------------------------------------------------------------------------------------------------

def _rank_entry(rank: int, world: int, port: int, target, payload):
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    rc = target(payload)
    if rc:
        raise SystemExit(rc)


def free_port() -> int:
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_ranks(world: int, target, payload) -> int:
    """Run target(payload) in `world` processes with RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* set as torchrun
    would (rendezvous on 127.0.0.1).  Raises if a rank fails."""
    import torch.multiprocessing as mp
    mp.spawn(_rank_entry, args=(world, free_port(), target, payload), nprocs=world, join=True)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="both", choices=["both", "f64", "f32"],
                    help="both (default): FP64 is the headline line, FP32 the block \"fp32\" of the same line")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1 only. weak: one image per GPU; strong: one image shared by the GPUs (tiles of 4096 rays)")
    ap.add_argument("--form", default="affine", choices=["affine", "coordtime", "bl"],
                    help="affine: gray2_integrate (eq. 13-14); coordtime: gray2_integrate_coordtime (eq. 18); "
                         "bl: gray2_integrate on Boyer-Lindquist states (eq. 1; the paper's Table 2 BL rows)")
    ap.add_argument("--workload", default="cfg3", choices=["cfg1", "cfg2", "cfg3", "cfg5"])
    ap.add_argument("--oracle-side", type=int, default=128, help="oracle sample: side x side rays of the same field of view")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--blocks", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-both", action="store_true", help="skip the two-precisions-at-once leg of --dtype both")
    ap.add_argument("--e2e-chunks", type=int, default=32, help="end-to-end leg: chunks pipelined over the streams")
    ap.add_argument("--e2e-streams", type=int, default=8, help="end-to-end leg: number of streams the chunks alternate between")
    args = ap.parse_args(argv)
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the ranks here
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit("bench.py: --gpus %d needs %d CUDA devices, this box has %d (the product path has no CPU "
                             "fallback and ranks do not share a GPU)" % (args.gpus, args.gpus, have))
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # keep the communicator log (nranks) on stderr
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        return launch_ranks(args.gpus, run_gpu, args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
