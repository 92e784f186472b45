"""Run the five BASELINE.json configs on the GPU and print one JSON report (GPU-only statistics).

    python report.py [--configs 1,2,3,4,5] [--cfg4-steps 100000] [--cfg4-n 1048576]

What each config asks to be reported (BASELINE.json "configs"):
  cfg1  Schwarzschild 64x64 image + 16 time-like orbits: status counts, step counts, invariant drift
  cfg2  Kerr a=0.99 512x512: status counts; the critical band is reported as the rays with unusually long paths
  cfg3  Kerr a=0.9375 1024x1024 in FP64 and FP32: FP32-vs-FP64 error on final (r, theta, phi) of escaped
        rays and on the capture mask
  cfg4  1,048,576 bound particles, fixed step 0.5, 100,000 steps: drift of E, L_z, Q and u.u
  cfg5  Kerr a=0.5 4096x4096 in FP32 and FP64: throughput under divergence in path length
The oracle comparisons live in tests/ (this script never touches the oracle).  It is harness, like bench.py: it sits beside it, outside the library package.
"""
from __future__ import annotations

import argparse
import json
import math
import time

import torch

import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from paper_1706_07062_b200 import gray2, inputs  # noqa: E402

INF = float("inf")


def _timed(fn):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    out = fn()
    e1.record()
    e1.synchronize()
    return out, e0.elapsed_time(e1) * 1e-3


def run_image(cfg, prec):
    sc = gray2.step_control(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                            capture_factor=cfg.capture_factor)
    st = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
    inv0 = gray2.invariants(st)
    stats = gray2.new_stats()
    gray2.integrate(st, INF, sc, stats=stats)          # warm-up launch on a copy would double memory: time a rerun
    torch.cuda.synchronize()
    st2 = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec, out=st)
    _, dt = _timed(lambda: gray2.integrate(st2, INF, sc, stats=stats))
    inv1 = gray2.invariants(st2)
    sd = gray2.stats_dict(stats)
    # the same image once more, scheduled longest first with the step counts of the trace above as the hint
    # (gray2_order_longest_first: what a caller that traces the same geometry repeatedly can do); same outputs
    st3 = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
    st3.order = gray2.order_longest_first(st2.nsteps)
    _, dt_lf = _timed(lambda: gray2.integrate(st3, INF, sc))
    identical = bool(torch.equal(st3.q, st2.q) and torch.equal(st3.nsteps, st2.nsteps))
    del st3
    ns = st2.nsteps
    esc = st2.status == gray2.ESCAPED
    rep = dict(sd, rays=cfg.n, seconds=dt, steps_per_s=sd["steps"] / dt,
               seconds_longest_first=dt_lf, steps_per_s_longest_first=sd["steps"] / dt_lf, longest_first_outputs_identical=identical,
               nsteps_min=int(ns.min()), nsteps_mean=float(ns.float().mean()), nsteps_max=int(ns.max()),
               captured_fraction=sd["n_captured"] / cfg.n,
               long_path_rays=int((ns > 1.5 * ns.float().mean()).sum()),
               max_abs_norm_escaped=float(inv1[3][esc].abs().max()),
               max_drift_E_escaped=float((inv1[0] - inv0[0])[esc].abs().max()),
               max_drift_Lz_escaped=float((inv1[1] - inv0[1])[esc].abs().max()),
               max_drift_Q_escaped=float((inv1[2] - inv0[2])[esc].abs().max()))
    return st2, rep


def spherical(q, a_eff):
    """KS r, theta, phi of positions q[1:4] (torch, double): x + i y = (r + i a) sin(theta) e^{i phi}."""
    x, y, z = q[1].double(), q[2].double(), q[3].double()
    w = x * x + y * y + z * z - a_eff * a_eff
    r = torch.sqrt(0.5 * (w + torch.sqrt(w * w + 4 * a_eff * a_eff * z * z)))
    th = torch.acos(torch.clamp(z / r, -1.0, 1.0))
    ph = torch.atan2(y, x) - torch.atan2(torch.full_like(r, a_eff), r)
    return r, th, ph


def compare_f32_f64(s64, s32, cfg):
    both_esc = (s64.status == gray2.ESCAPED) & (s32.status == gray2.ESCAPED)
    same = both_esc & (s64.nsteps == s32.nsteps)
    ra, ta, pa = spherical(s64.q, s64.a_eff)
    rb, tb, pb = spherical(s32.q, s32.a_eff)
    dphi = torch.remainder(pb - pa + math.pi, 2 * math.pi) - math.pi
    err = {"r_rel": ((rb - ra).abs() / ra)[same], "theta": (tb - ta).abs()[same], "phi": dphi.abs()[same]}
    qs = torch.tensor([0.5, 0.9, 0.99, 0.999, 1.0], dtype=torch.float64, device="cuda")

    def quant(v):
        v = v.double()
        k = (qs * (v.numel() - 1)).long()
        return [float(x) for x in torch.sort(v).values[k]]

    # direction of the spatial velocity at the stopping state: insensitive to a +-1 step difference
    va = s64.q[5:8].double()
    vb = s32.q[5:8].double()
    cosang = (va * vb).sum(0) / (va.norm(dim=0) * vb.norm(dim=0))
    ang = torch.acos(torch.clamp(cosang, -1.0, 1.0))[both_esc]
    mask_diff = int(((s64.status == gray2.CAPTURED) != (s32.status == gray2.CAPTURED)).sum())
    return {"escaped_in_both": int(both_esc.sum()), "equal_step_count_fraction": float(same.sum()) / max(int(both_esc.sum()), 1),
            "quantiles": [0.5, 0.9, 0.99, 0.999, 1.0],
            "final_r_relative": quant(err["r_rel"]), "final_theta_rad": quant(err["theta"]),
            "final_phi_rad": quant(err["phi"]), "velocity_direction_rad_all_escaped": quant(ang),
            "rays_beyond_1e-4_in_r_theta_or_phi": int(((err["r_rel"] > 1e-4) | (err["theta"] > 1e-4) | (err["phi"] > 1e-4)).sum()),
            "capture_mask_disagreements": mask_diff, "rays": cfg.n}


def report_cfg3():
    """BASELINE.json configs[2]: FP32-vs-FP64 error on the final (r, theta, phi) of escaped rays and on the capture
    mask.  Twice: (i) each precision from its own gray2_init_null (the float image differs from the double one by
    the rounding of the starting points, ~3e-5 M at r_obs = 1000 M), (ii) the double run started from the float
    initial state, so that only the arithmetic of the integration differs."""
    cfg = inputs.CFG3_NULL
    s64, r64 = run_image(cfg, gray2.F64)
    s32, r32 = run_image(cfg, gray2.F32)
    out = {"f64": r64, "f32": r32, "fp32_vs_fp64": compare_f32_f64(s64, s32, cfg)}
    del s64
    i32 = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=gray2.F32)
    w = gray2.State(i32.n, gray2.F64, i32.q.double(), i32.lam.clone(), i32.status.clone(), i32.nsteps.clone(),
                    i32.a_eff, i32.kind, i32.reversed, i32.coords)
    del i32
    sc = gray2.step_control(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                            capture_factor=cfg.capture_factor)
    gray2.integrate(w, INF, sc)
    out["fp32_vs_fp64_same_float_inputs"] = compare_f32_f64(w, s32, cfg)
    return out


def report_cfg1():
    _, img = run_image(inputs.CFG1_NULL, gray2.F64)
    xu8, r0 = inputs.cfg1_orbits()
    st = gray2.init_timelike(0.0, xu8)
    inv0 = gray2.invariants(st)
    stats = gray2.new_stats()
    gray2.integrate(st, INF, gray2.step_control(mode=0, h_fixed=0.5, max_steps=5000), stats=stats)
    inv1 = gray2.invariants(st)
    r = spherical(st.q, 0.0)[0].cpu()
    orb = dict(gray2.stats_dict(stats), max_abs_r_minus_r0=float((r - torch.tensor(r0)).abs().max()),
               max_drift=[float((b - a_).abs().max()) for a_, b in zip(inv0, inv1)])
    return {"image": img, "orbits": orb}


def report_cfg4(n, nsteps):
    t0 = time.time()
    xu8, meta = inputs.cfg4_ensemble(n)
    gen_s = time.time() - t0
    st = gray2.init_timelike(0.7, xu8)
    inv0 = gray2.invariants(st)
    stats = gray2.new_stats()
    sc = gray2.step_control(mode=0, h_fixed=0.5, max_steps=nsteps)
    _, dt = _timed(lambda: gray2.integrate(st, INF, sc, stats=stats))
    inv1 = gray2.invariants(st)
    sd = gray2.stats_dict(stats)
    names = ("E", "Lz", "Q", "norm")
    drift = {}
    alive = st.status == gray2.MAXSTEPS     # a few marginal orbits plunge at this step size; they end inside 1.01 r_plus
    for nm, a_, b in zip(names, inv0, inv1):
        d = (b - a_)[alive]
        rel = d / torch.clamp(a_[alive].abs(), min=1.0)
        drift[nm] = {"max_abs": float(d.abs().max()), "rms": float(d.pow(2).mean().sqrt()),
                     "max_rel_to_max(1,|value|)": float(rel.abs().max())}
    return dict(sd, particles=n, steps_per_particle=nsteps, seconds=dt, steps_per_s=sd["steps"] / dt,
                generator_seconds=gen_s, acceptance=meta["acceptance"], drift_of_particles_still_orbiting=drift)


def report_paper_benchmark():
    """The paper's own benchmark shape: null geodesics traced back from an image at
    r = 1024 M toward a = 0.999, fixed step, 1024 RK4 steps per call, calls repeated until every ray is
    captured or has escaped beyond its initial radius, in both coordinate systems of Table 2 (KS: eq. 13-14,
    BL: eq. 1 through gray2_convert); image sizes 64^2 ... 1024^2; reported: the
    shortest call time divided by the steps it executed = ns per RK4 step per ray (Table 2's unit).
    The paper does not state step size, inclination or field of view: h = 1/32 (64 calls x 1024 steps
    cover the 2 x 1024 M path), i = 60 deg, +-15 M are used here."""
    out = {}
    for coords, cname in ((gray2.KS, "KS"), (gray2.BL, "BL")):
        for prec, name in ((gray2.F64, "double"), (gray2.F32, "single")):
            best = {}
            for side in (64, 128, 256, 512, 1024):
                st = gray2.init_null(0.999, 1024.0, math.radians(60.0), 15.0, 15.0, side, side, prec=prec)
                if coords == gray2.BL:
                    st = gray2.convert(st, gray2.BL)
                stats = gray2.new_stats()
                calls, best_ns, total_steps = 0, float("inf"), 0
                while True:
                    calls += 1
                    sc = gray2.step_control(mode=0, h_fixed=1.0 / 32.0, r_escape=1024.5, max_steps=1024 * calls)
                    _, dt = _timed(lambda: gray2.integrate(st, INF, sc, stats=stats))
                    sd = gray2.stats_dict(stats)
                    total_steps += sd["steps"]
                    if sd["steps"] > 0.5 * 1024 * side * side:           # launches that still step most rays
                        best_ns = min(best_ns, 1e9 * dt / sd["steps"])
                    if sd["n_maxsteps"] == 0 or calls >= 80:
                        break
                    st.status[st.status == gray2.MAXSTEPS] = gray2.ACTIVE   # continue the unfinished rays
                best[str(side)] = {"calls": calls, "best_ns_per_step_per_ray": best_ns, "total_steps": total_steps}
            out[cname + "_" + name] = {"per_image_size": best,
                                       "ns_per_step_per_ray": min(v["best_ns_per_step_per_ray"] for v in best.values())}
    out["paper_table2_SoA_best"] = {"KS_single": "0.309 ns", "KS_double": "1.15 ns", "BL_single": "0.175 ns",
                                    "BL_double": "1.66 ns", "device": "Titan Black", "cite": "PAPER.md:283-288"}
    return out


def report_bl_vs_ks():
    """The same images traced in both coordinate systems (PAPER.md:49-51 made quantitative): how many rays
    end with a different fate in Boyer-Lindquist coordinates, and where they are (all of them graze the
    axis: |L_z|/E small), per image config, FP64.  Kerr-Schild is the reference: tests/ pin it to Carter's
    potential on every ray outside the critical band."""
    out = {}
    for cfg in (inputs.CFG1_NULL, inputs.CFG2_NULL, inputs.CFG3_NULL, inputs.CFG5_NULL):
        sc = gray2.step_control(mode=1, eta=cfg.eta, r_escape=cfg.r_escape, max_steps=cfg.max_steps,
                                capture_factor=cfg.capture_factor)
        ks = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
        E, Lz, Q, _ = gray2.invariants(ks)
        bl = gray2.convert(ks, gray2.BL)
        sk, sb = gray2.new_stats(), gray2.new_stats()
        _, tk = _timed(lambda: gray2.integrate(ks, INF, sc, stats=sk))
        _, tb = _timed(lambda: gray2.integrate(bl, INF, sc, stats=sb))
        differ = ks.status != bl.status
        esc = (ks.status == gray2.ESCAPED) & ~differ
        late = esc & ((ks.nsteps - bl.nsteps).abs() > 1)
        xi = (Lz / E).abs()
        out[cfg.name] = {
            "rays": cfg.n, "ks": gray2.stats_dict(sk), "bl": gray2.stats_dict(sb),
            "ks_steps_per_s": gray2.stats_dict(sk)["steps"] / tk, "bl_steps_per_s": gray2.stats_dict(sb)["steps"] / tb,
            "rays_with_different_fate": int(differ.sum()), "fraction": float(differ.float().mean()),
            "escaped_rays_with_step_count_off_by_more_than_1": int(late.sum()),
            "max_abs_Lz_over_E_of_those_rays": float(xi[differ | late].max()) if bool((differ | late).any()) else None,
            "median_abs_Lz_over_E_of_all_rays": float(xi.median()),
        }
        del ks, bl
        torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", default="1,2,3,4,5", help="comma list of 1..5, P (the paper's benchmark shape), B (Boyer-Lindquist vs Kerr-Schild images)")
    ap.add_argument("--cfg4-steps", type=int, default=100000)
    ap.add_argument("--cfg4-n", type=int, default=1 << 20)
    args = ap.parse_args()
    want = set(args.configs.split(","))
    out = {"device": torch.cuda.get_device_name(0), "library": gray2.version()}
    if "1" in want:
        out["cfg1"] = report_cfg1()
    if "2" in want:
        out["cfg2"] = {"f64": run_image(inputs.CFG2_NULL, gray2.F64)[1]}
    if "3" in want:
        out["cfg3"] = report_cfg3()
    if "4" in want:
        out["cfg4"] = report_cfg4(args.cfg4_n, args.cfg4_steps)
    if "5" in want:
        out["cfg5"] = {"f32": run_image(inputs.CFG5_NULL, gray2.F32)[1]}
        torch.cuda.empty_cache()
        out["cfg5"]["f64"] = run_image(inputs.CFG5_NULL, gray2.F64)[1]
    if "P" in want:
        out["paper_benchmark"] = report_paper_benchmark()
    if "B" in want:
        out["bl_vs_ks"] = report_bl_vs_ks()
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
