#!/usr/bin/env python
"""bench.py -- geodesic RK4 steps/s of the whole hot path on BASELINE.json's headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--workload cfg3|cfg1|cfg2|cfg5]
    python bench.py --impl reference ...      # the oracle, as it stands, on the host cores

A "step" is one pass of the whole path over one batch: gray2_init_null (image-plane initial conditions)
-> gray2_integrate (fused RHS + RK4 + termination + refill) -> gray2_invariants, on the 1024 x 1024
Kerr image of BASELINE.json configs[2] ("cfg3": a = 0.9375, r_obs = 1000 M, i = 60 deg, +-15 M), which is
the workload north_star quotes the target on.  The metric is geodesic RK4 steps per second (whole job,
summed over ranks; each rank traces its own image: weak scaling, no collective on the data path;
--scaling strong shares ONE image among the ranks in tiles of 4096 rays, again without a collective).

One JSON line is printed by rank 0; see DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
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

# DRAM traffic of the dominant kernel, dram__bytes_read.sum + dram__bytes_write.sum per launch, from the
# `ncu --set full` captures summarised in profiles/r01_ncu_integrate_f{64,32}_v4.txt (cfg3, affine form) and
# profiles/r01_ncu_integrate_bl_f{64,32}.txt (cfg3, Boyer-Lindquist form).
# Algorithmic state traffic is 2 x 80 B (FP64) or 2 x 48 B (FP32) per ray.
NCU_DRAM_BYTES = {("cfg3", "f64", "affine"): 83935744 + 31088896, ("cfg3", "f32", "affine"): 50348544 + 1701632,
                  ("cfg3", "f64", "bl"): 83937280 + 34206208, ("cfg3", "f32", "bl"): 50350080 + 1716480}


def nominal_peak_tflops(dtype: str, n_sms: int, sm_max_mhz: float) -> float:
    return n_sms * FP_LANES[dtype] * 2.0 * sm_max_mhz * 1e6 / 1e12


def load_measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons (profiling recipe).  It is started before the warm-up
    so that nvidia-smi's start-up cost is not inside the timed region; every sample is stamped on arrival
    and only the samples that fall inside the timed window are reported."""
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

    def stop(self, t_begin, t_end) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.05)
        self.proc.terminate()
        sm, smax, power, reasons = [], [], [], set()
        for stamp, ln in self.samples:
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


def workload_config(name: str):
    from paper_1706_07062_b200 import inputs
    return {"cfg1": inputs.CFG1_NULL, "cfg2": inputs.CFG2_NULL, "cfg3": inputs.CFG3_NULL,
            "cfg5": inputs.CFG5_NULL}[name]


# ---------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle, as it stands, on the host cores, on a bounded sample
# ---------------------------------------------------------------------------------------------------

def oracle_sample_config(cfg, side: int):
    return cfg.scaled(side)


def time_oracle(cfg, side: int, steps: int, warmup: int):
    """Each step = init_null + integrate + invariants of the workload's field of view sampled on side^2 rays."""
    import oracle
    sub = oracle_sample_config(cfg, side)
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

def run_gpu(args):
    import torch
    import torch.distributed as dist

    from paper_1706_07062_b200 import gray2

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:                       # in-tree build (a no-op when libgray2.so is up to date)
        from paper_1706_07062_b200 import build as _build
        _build.build()
    if world > 1:
        dist.barrier()
    gray2.load_library()

    cfg = workload_config(args.workload)
    prec = gray2.F64 if args.dtype == "f64" else gray2.F32
    coord = args.form == "coordtime"
    bl = args.form == "bl"          # Boyer-Lindquist variant (Table 2 "BL" rows): init -> convert -> integrate
    flops_per_step = (gray2.flops_per_step_coordtime(prec) if coord else
                      gray2.flops_per_step_bl(prec) if bl else gray2.flops_per_step(prec))
    integrate = gray2.integrate_coordtime if coord else gray2.integrate
    props = torch.cuda.get_device_properties(local)
    n_sms = props.multi_processor_count
    peaks = load_measured_peaks()
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    if args.threads or args.blocks:
        gray2.set_launch(prec, args.threads, args.blocks)

    sc = gray2.step_control(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                            capture_factor=cfg.capture_factor)
    # --scaling strong: ONE image shared by all ranks, rays dealt out in tiles of 4096;
    # weak (default): every rank traces its own image.  Neither has a collective on the data path.
    strong = args.scaling == "strong" and world > 1
    n_local = gray2.shard_count(cfg.n, SHARD_TILE, rank, world) if strong else cfg.n
    st = gray2.State.empty(n_local, prec)
    st_ks = gray2.State.empty(n_local, prec) if bl else st
    stats = gray2.new_stats()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    def one_step(ev=None):
        if ev: ev[0].record(stream)
        if strong:
            gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, SHARD_TILE,
                                  rank, world, prec=prec, out=st_ks)
        else:
            gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec, out=st_ks)
        if bl: gray2.convert(st_ks, gray2.BL, out=st)
        if ev: ev[1].record(stream)
        integrate(st, INF, sc, stats=stats)
        if ev: ev[2].record(stream)
        inv = gray2.invariants(st)
        if ev: ev[3].record(stream)
        return inv

    try:
        gpu_id = "GPU-" + str(props.uuid) if not str(props.uuid).startswith("GPU-") else str(props.uuid)
    except Exception:
        gpu_id = str(local)
    sampler = ClockSampler(gpu_id)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        one_step()
    torch.cuda.synchronize()
    sampler.wait_for_first_sample()

    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t_window0 = time.perf_counter()
    t_step, t_int, steps_total = 0.0, 0.0, 0
    for _ in range(args.steps):
        flush.fill_(1)                                     # flush L2 between timed iterations (untimed)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        one_step(ev)
        ev[3].synchronize()
        t_step += ev[0].elapsed_time(ev[3]) * 1e-3
        t_int += ev[1].elapsed_time(ev[2]) * 1e-3
        steps_total += int(stats[0].item())
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop(t_window0, time.perf_counter())

    # ---- end to end through the public API with HOST buffers (pinned): H2D of the 8-vectors, D2H of results
    host_in = torch.empty((n_local, 8), dtype=torch.float64).pin_memory()
    if strong:
        src = gray2.init_null_shard(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, SHARD_TILE,
                                    rank, world, prec=gray2.F64)
    else:
        src = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=gray2.F64)
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
                if bl:
                    ks = parts_ks[c]
                    gray2.init_timelike(a_eff, host_in_np[lo:hi], prec=prec, out=ks)
                    ks.kind, ks.reversed = gray2.NULL, 1
                    gray2.convert(ks, gray2.BL, out=part)
                else:
                    gray2.init_timelike(a_eff, host_in_np[lo:hi], prec=prec, out=part)   # H2D inside (explicit 8-vectors)
                    part.kind, part.reversed = gray2.NULL, 1
                integrate(part, INF, sc, stats=chunk_stats[c])
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
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e2e_steps = sum(e2e_step() for _ in range(e2e_n))
    t_e2e = time.perf_counter() - t0

    # ---- FMA-only probes of the pipe at the clocks of the moment (context for the nominal peak)
    scratch = torch.zeros(8, dtype=torch.float64 if prec == gray2.F64 else torch.float32, device="cuda")
    iters = 20000 if prec == gray2.F64 else 40000
    probe = {}
    for name, regs in (("imm", 0), ("regs", 1), ("fresh", 2)) + ((("packed", 3),) if prec == gray2.F32 else ()):
        gray2.fma_probe(prec, n_sms * 8, 256, iters, scratch, register_operands=regs)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        probe_flops = gray2.fma_probe(prec, n_sms * 8, 256, iters, scratch, register_operands=regs)
        e1.record(stream)
        e1.synchronize()
        probe[name] = probe_flops / (e0.elapsed_time(e1) * 1e-3) / 1e12
    fma_probe_tflops = probe["imm"]

    # ---- reduce over ranks: time = max, work = sum
    from paper_1706_07062_b200 import multi
    (t_step, t_int, t_e2e), (steps_all, e2e_all) = multi.reduce_job([t_step, t_int, t_e2e], [steps_total, e2e_steps],
                                                                    device="cuda")

    if rank == 0:
        value = steps_all / t_step
        peak = nominal_peak_tflops(args.dtype, n_sms, sm_max_mhz)
        achieved = (steps_total * flops_per_step / t_int) / 1e12          # this rank's dominant kernel
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_step / args.steps, "higher_is_better": True,
            "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": cfg.name, "rays_per_gpu": n_local, "rk4_steps_per_pass": steps_total // args.steps,
                       "a": cfg.a, "r_obs": cfg.r_obs, "inclination_deg": cfg.inclination_deg, "fov_half": cfg.fov,
                       "form": args.form, "step_rule": ("dt = %g r" if coord else "dlambda = %g r") % cfg.eta, "l2": "flushed between timed iterations (256 MiB fill)",
                       "parallelism": ("one image dealt out in tiles of %d rays, no collective" % SHARD_TILE) if strong
                                      else "independent image per GPU, no collective"},
            "clocks": clocks,
            "e2e": {"value": e2e_all / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "api": "gray2_init_timelike(host 8-vectors) -> %sgray2_integrate -> gray2_invariants -> D2H of state, invariants, stats" % ("gray2_convert -> " if bl else ""),
                    "chunks": n_chunks, "streams": n_streams},
            "gpu_launches": (5 if bl else 4) * args.steps,
            "roofline": {"bound": "alu", "kernel": ("integrate_kernel<double%s>" if prec == gray2.F64 else "integrate_kernel_f32x2<%s>") % (
                             ", coordinate time" if coord else ", Boyer-Lindquist" if bl else ("" if prec == gray2.F64 else "affine")),
                         "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": NCU_DRAM_BYTES.get((args.workload, args.dtype, args.form)),
                         "traffic_unit": "bytes per launch (ncu, profiles/r01_ncu_integrate_*.txt)",
                         "flops_per_rk4_step": flops_per_step,
                         "kernel_ms": 1e3 * t_int / args.steps, "kernel_share_of_step": t_int / t_step,
                         "peak_source": "nominal: %d SMs x %d lanes x 2 x %.0f MHz" % (n_sms, FP_LANES[args.dtype], sm_max_mhz),
                         "fma_probe_tflops": fma_probe_tflops, "frac_of_fma_probe": achieved / fma_probe_tflops,
                         "fma_probe_register_operands_tflops": probe["regs"],
                         "fma_probe_fresh_register_operands_tflops": probe["fresh"],
                         "fma_probe_packed_fp32x2_tflops": probe.get("packed")},
        }
        if not args.no_cpu_baseline and world == 1:
            # a first pass on oracle_side^2 rays sizes the sample: about 12 s of wall clock on this box's cores
            _, s_probe, _, _ = time_oracle(cfg, args.oracle_side, 1, 0)
            side = int(args.oracle_side * math.sqrt(max(1.0, 12.0 / max(s_probe, 1e-3)))) // 32 * 32
            side = max(args.oracle_side, min(side, 512, cfg.nx))
            v, s_per, cores, sub = time_oracle(cfg, side, 1, 0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": "%s field of view on %dx%d rays, one pass (%.1f s)" % (
                                        args.workload, side, side, s_per)}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
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
    ap.add_argument("--e2e-chunks", type=int, default=32, help="end-to-end leg: chunks pipelined over the streams")
    ap.add_argument("--e2e-streams", type=int, default=8, help="end-to-end leg: number of streams the chunks alternate between")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
