"""GPU edge cases and full-size checks: ragged and tiny batches, resume, idempotence, INVALID rays,
max_steps, determinism across launch shapes, and sampled parity at BASELINE.json's full sizes in the
launch configuration bench.py times."""
import numpy as np
import pytest
import torch

import image_helpers as ih
import oracle
from gpu_helpers import (INF, TOL_STATE_F32, TOL_STATE_F64, TWINS_ORBIT, accumulated_rounding_f64, assert_fp32_parity, image_sc, image_sc_kw, make_straddle_check, run_gpu_image,
                         sc_pair, state_rel_error, take, to_oracle_state, twin_sensitivity)
from paper_1706_07062_b200 import gray2, inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("nx,ny", [(1, 1), (5, 1), (31, 1), (33, 3), (129, 1)])
def test_tiny_and_ragged_batches(nx, ny):
    cfg = inputs.NullImageConfig("t", 0.9, 200.0, 40.0, 7.0, nx, ny, r_escape=250.0)
    g0, g, gstats = run_gpu_image(cfg)
    o = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, nx, ny)
    ostats = oracle.integrate(o, INF, image_sc(cfg)[1])
    gst = to_oracle_state(g)
    assert np.array_equal(gst.status, o.status) and np.array_equal(gst.nsteps, o.nsteps)
    assert state_rel_error(gst.q, o.q, o.a_eff).max() < TOL_STATE_F64
    assert gstats == ostats


def test_partial_n_leaves_the_rest_untouched():
    cfg = inputs.CFG1_NULL
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    before = g.clone()
    stats = gray2.new_stats()
    gray2.integrate(g, INF, image_sc(cfg)[0], n=1000, stats=stats)
    torch.cuda.synchronize()
    assert torch.equal(g.q[:, 1000:], before.q[:, 1000:]) and (g.status[1000:] == gray2.ACTIVE).all()
    assert (g.status[:1000] != gray2.ACTIVE).all()
    sd = gray2.stats_dict(stats)
    assert sd["n_captured"] + sd["n_escaped"] == 1000 and sd["steps"] == int(g.nsteps[:1000].sum().item())


def test_resume_and_idempotence():
    cfg = inputs.CFG3_NULL.scaled(40)
    gsc, osc = image_sc(cfg)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    s1 = gray2.new_stats()
    gray2.integrate(g, 900.0, gsc, stats=s1)         # every ray is still far out: stays ACTIVE, lambda = 900
    oracle.integrate(o, 900.0, osc)
    gst = to_oracle_state(g)
    assert (gst.status == gray2.ACTIVE).all() and np.allclose(gst.lam, 900.0, atol=1e-9)
    assert np.array_equal(gst.nsteps, o.nsteps)
    assert state_rel_error(gst.q, o.q, o.a_eff).max() < TOL_STATE_F64
    assert gray2.stats_dict(s1)["n_active"] == cfg.n
    gray2.integrate(g, INF, gsc, stats=s1)
    oracle.integrate(o, INF, osc)
    gst = to_oracle_state(g)
    d, _ = ih.classify_image(cfg, oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny))
    outside = d > 1e-3
    assert np.array_equal(gst.status[outside], o.status[outside]) and np.array_equal(gst.nsteps[outside], o.nsteps[outside])
    # a second identical call is a no-op
    snap = g.clone()
    s2 = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=s2)
    torch.cuda.synchronize()
    assert torch.equal(snap.q, g.q) and torch.equal(snap.nsteps, g.nsteps) and torch.equal(snap.lam, g.lam)
    assert gray2.stats_dict(s2)["steps"] == 0 and gray2.stats_dict(s2)["n_active"] == 0


def test_invalid_rays_are_data_not_errors():
    cfg = inputs.CFG1_NULL.scaled(16)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    g.q[5, 3] = float("nan")
    g.q[2, 7] = float("inf")
    g.q[0, 9] = float("nan")
    stats = gray2.new_stats()
    gray2.integrate(g, INF, image_sc(cfg)[0], stats=stats)
    sd = gray2.stats_dict(stats)
    st = g.status.cpu().numpy()
    assert st[3] == gray2.INVALID and st[7] == gray2.INVALID and st[9] == gray2.INVALID
    assert g.nsteps[3].item() == 0 and sd["n_invalid"] == 3 and sd["n_active"] == 0
    assert sd["n_captured"] + sd["n_escaped"] == cfg.n - 3


def test_max_steps_is_absolute_and_fixed_step_lambda():
    xu8, _ = inputs.cfg4_ensemble(300)
    g = gray2.init_timelike(0.7, xu8)
    o = oracle.init_timelike(0.7, xu8)
    gsc, osc = sc_pair(mode=0, h_fixed=0.5, max_steps=700)
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    oracle.integrate(o, INF, osc)
    gst = to_oracle_state(g)
    assert (gst.nsteps == 700).all() and (gst.status == gray2.MAXSTEPS).all() and np.allclose(gst.lam, 350.0)
    assert state_rel_error(gst.q, o.q, 0.7).max() < TOL_STATE_F64
    assert gray2.stats_dict(stats)["steps"] == 300 * 700
    # raising the budget continues from where it stopped
    g.status.fill_(gray2.ACTIVE)
    gsc2, _ = sc_pair(mode=0, h_fixed=0.5, max_steps=1000)
    gray2.integrate(g, INF, gsc2, stats=stats)
    assert (g.nsteps == 1000).all() and gray2.stats_dict(stats)["steps"] == 300 * 300


def test_results_do_not_depend_on_launch_shape_or_run():
    cfg = inputs.CFG3_NULL.scaled(150, 90)
    ref = None
    try:
        for shape in [(0, 0), (128, 4), (64, 6), (0, 0)]:
            gray2.set_launch(gray2.F64, *shape)
            _, g, stats = run_gpu_image(cfg)
            cur = (g.q.clone(), g.nsteps.clone(), g.status.clone(), g.lam.clone(), stats)
            if ref is None:
                ref = cur
            else:
                assert all(torch.equal(x, y) for x, y in zip(ref[:4], cur[:4])) and ref[4] == cur[4]
    finally:
        gray2.set_launch(gray2.F64, 0, 0)


def test_fp32_packed_and_scalar_kernels_agree_bit_for_bit():
    """FP32 runs two geodesics per thread with packed FP32x2 instructions by default; the one-per-thread
    float kernel must give the same bits (every FMA is explicit, the library is built with --fmad=false)."""
    cfg = inputs.CFG3_NULL.scaled(150, 91)          # odd ray count: the last thread has an empty second slot
    ref = None
    try:
        for shape in [(0, 0), (256, 2), (256, 1), (128, 3), (128, 4), (128, 8), (128, 6)]:
            gray2.set_launch(gray2.F32, *shape)
            _, g, stats = run_gpu_image(cfg, prec=gray2.F32)
            cur = (g.q.clone(), g.nsteps.clone(), g.status.clone(), g.lam.clone(), stats)
            if ref is None:
                ref = cur
            else:
                assert all(torch.equal(x, y) for x, y in zip(ref[:4], cur[:4])) and ref[4] == cur[4], shape
    finally:
        gray2.set_launch(gray2.F32, 0, 0)
    assert ref[4]["n_active"] == 0 and ref[4]["n_captured"] + ref[4]["n_escaped"] == cfg.n


def test_concurrent_calls_on_two_streams():
    """Two integrations in flight at once on different streams (each takes its own work-queue slot) give
    the same bits as the same calls issued one after the other."""
    cfgs = [inputs.CFG3_NULL.scaled(96), inputs.CFG2_NULL.scaled(80)]
    serial = []
    for cfg in cfgs:
        _, g, stats = run_gpu_image(cfg)
        serial.append((g.q.clone(), g.nsteps.clone(), stats))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    states, stats_t = [], []
    torch.cuda.synchronize()
    for cfg, stream in zip(cfgs, streams):
        with torch.cuda.stream(stream):
            g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, stream=stream)
            st = gray2.new_stats()
            gray2.integrate(g, INF, image_sc(cfg)[0], stats=st, stream=stream)
            states.append(g)
            stats_t.append(st)
    torch.cuda.synchronize()
    for (q, ns, sd), g, st in zip(serial, states, stats_t):
        assert torch.equal(q, g.q) and torch.equal(ns, g.nsteps) and gray2.stats_dict(st) == sd


def test_more_calls_in_flight_than_work_queue_slots():
    """The library has 64 work-queue slots per device.  160 integrations enqueued without a synchronise on
    four streams (slots are reused while earlier users may still run: the reuse waits on the device) give the
    bits of the same image integrated alone."""
    cfg = inputs.CFG3_NULL.scaled(48)
    _, ref, ref_stats = run_gpu_image(cfg)
    streams = [torch.cuda.Stream() for _ in range(4)]
    runs = []
    torch.cuda.synchronize()
    for i in range(160):
        stream = streams[i % 4]
        with torch.cuda.stream(stream):
            g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, stream=stream)
            st = gray2.new_stats()
            gray2.integrate(g, INF, image_sc(cfg)[0], stats=st, stream=stream)
            runs.append((g, st))
    torch.cuda.synchronize()
    for g, st in runs:
        assert torch.equal(ref.q, g.q) and torch.equal(ref.nsteps, g.nsteps) and torch.equal(ref.status, g.status)
        assert gray2.stats_dict(st) == ref_stats


def test_set_launch_may_race_with_integrations():
    """gray2.h: any number of host threads may call in.  One thread keeps switching the launch shape among the
    compiled variants while four others integrate: no call may fail ("no compiled variant" would be a torn read
    of the pair) and every result equals the reference bit for bit."""
    import threading
    cfg = inputs.CFG3_NULL.scaled(96, 64)
    gsc, _ = image_sc(cfg)
    ref = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    gray2.integrate(ref, INF, gsc)
    torch.cuda.synchronize()
    stop, errors = threading.Event(), []

    def switcher():
        shapes = [(128, 3), (128, 4), (64, 6), (256, 1), (128, 2), (0, 0)]
        k = 0
        while not stop.is_set():
            gray2.set_launch(gray2.F64, *shapes[k % len(shapes)])
            k += 1

    def worker():
        try:
            stream = torch.cuda.Stream()
            for _ in range(12):
                with torch.cuda.stream(stream):
                    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, stream=stream)
                    gray2.integrate(g, INF, gsc, stream=stream)
                stream.synchronize()
                assert torch.equal(g.q, ref.q) and torch.equal(g.nsteps, ref.nsteps) and torch.equal(g.status, ref.status)
        except Exception as exc:          # noqa: BLE001
            errors.append(exc)

    sw = threading.Thread(target=switcher)
    sw.start()
    ws = [threading.Thread(target=worker) for _ in range(4)]
    for w in ws: w.start()
    for w in ws: w.join()
    stop.set()
    sw.join()
    gray2.set_launch(gray2.F64, 0, 0)
    assert not errors, errors


def test_init_explicit_from_four_threads_with_growing_batches():
    """Any number of host threads (include/gray2.h "Threads"): four threads, a stream each, feed batches that keep
    outgrowing their staging buffers, so that one thread's cudaFree + cudaMalloc runs while the others copy.  Every
    state must hold exactly the rows its own thread passed in."""
    import threading
    errors = []

    def worker(k):
        try:
            torch.cuda.set_device(0)
            stream = torch.cuda.Stream()
            rng = np.random.default_rng(100 + k)
            for rnd, n in enumerate((257, 4099, 1000, 20011, 65537, 3, 131101)):
                xu8 = rng.uniform(-40.0, 40.0, (n, 8))
                prec = gray2.F64 if (rnd + k) % 2 == 0 else gray2.F32
                with torch.cuda.stream(stream):
                    g = gray2.init_explicit(0.3, xu8, gray2.NULL, prec=prec, stream=stream)
                xu8_sent = xu8.copy()
                xu8[:] = 0.0                  # the host array may be reused as soon as the call returns
                stream.synchronize()
                want = torch.tensor(xu8_sent.T, device="cuda").to(g.q.dtype)
                if not torch.equal(g.q, want):
                    errors.append((k, n, "state differs"))
                if not bool((g.status == gray2.ACTIVE).all()) or not bool((g.nsteps == 0).all()):
                    errors.append((k, n, "status / nsteps"))
        except Exception as exc:              # noqa: BLE001 - reported by the main thread
            errors.append((k, repr(exc)))

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(4)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


def test_schedule_changes_no_output_bit():
    """gray2_state.order (optional order array): the longest-first order from a previous
    trace is a permutation sorted by decreasing step count, and integrating with it -- in both precisions, in
    the coordinate-time and Boyer-Lindquist forms -- gives the outputs of the unordered run bit for bit."""
    cfg = inputs.CFG3_NULL.scaled(160, 123)
    gsc, _ = image_sc(cfg)
    for prec in (gray2.F64, gray2.F32):
        for form in ("affine", "coordtime", "bl"):
            def fresh():
                g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
                return gray2.convert(g, gray2.BL) if form == "bl" else g
            run = gray2.integrate_coordtime if form == "coordtime" else gray2.integrate
            ref, sref = fresh(), gray2.new_stats()
            run(ref, INF, gsc, stats=sref)
            order = gray2.order_longest_first(ref.nsteps)
            o = order.cpu().numpy()
            assert np.array_equal(np.sort(o), np.arange(cfg.n))
            hint = ref.nsteps.cpu().numpy()[o].astype(np.int64)
            width = int(hint.max()) // 4096 + 1               # 4096 bins over [0, max]: sorted up to the bin width
            assert (np.diff((hint.max() - hint) // width) >= 0).all() and hint.max() - hint[0] < width
            g, sg = fresh(), gray2.new_stats()
            g.order = order
            run(g, INF, gsc, stats=sg)
            torch.cuda.synchronize()
            assert torch.equal(ref.q, g.q) and torch.equal(ref.nsteps, g.nsteps) and torch.equal(ref.status, g.status)
            assert torch.equal(ref.lam, g.lam) and torch.equal(sref, sg)
    # a call that covers only part of the state ignores the schedule (it would not be a permutation of that part)
    a = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    b = a.clone()
    b.order = order
    gray2.integrate(a, INF, gsc, n=1000)
    gray2.integrate(b, INF, gsc, n=1000)
    assert torch.equal(a.q, b.q) and torch.equal(a.status, b.status) and (b.status[1000:] == gray2.ACTIVE).all()
    # hints with a huge range (bins wider than one), zeros and negatives
    hint = torch.tensor([5, 0, -3, 2_000_000_000, 17, 17, 1_000_000], dtype=torch.int32, device="cuda")
    o = gray2.order_longest_first(hint).cpu().numpy()
    assert sorted(o.tolist()) == list(range(7)) and o[0] == 3 and o[1] == 6


def test_a_wrong_schedule_is_data_not_a_fault():
    """gray2_state.order that is not a permutation (include/gray2.h): entries outside 0..n-1 are passed over, a geodesic
    listed twice comes out with the bits of the unordered run, one listed nowhere is not touched and stays ACTIVE.
    Both precisions (the one-per-thread and the packed ordered kernels)."""
    cfg = inputs.CFG3_NULL.scaled(96, 64)
    gsc, _ = image_sc(cfg)
    n = cfg.n
    rng = np.random.default_rng(8)
    bad = rng.permutation(n).astype(np.int64)
    left_out = bad[:500].copy()                       # these 500 positions get other contents:
    bad[:100] = n + rng.integers(0, 1 << 20, 100)     #   beyond the end,
    bad[100:200] = -1 - rng.integers(0, 1 << 20, 100) #   negative,
    bad[200:300] = 0x7fffffff                         #   the largest int32,
    bad[300:500] = bad[500:700]                       #   and 200 geodesics listed twice
    listed = np.zeros(n, dtype=bool)
    listed[bad[(bad >= 0) & (bad < n)]] = True
    assert not listed[left_out].any() and listed.sum() == n - 500
    for prec in (gray2.F64, gray2.F32):
        ref = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
        g = ref.clone()
        start = ref.clone()
        gray2.integrate(ref, INF, gsc)
        g.order = torch.tensor(bad, dtype=torch.int32, device="cuda")
        stats = gray2.new_stats()
        gray2.integrate(g, INF, gsc, stats=stats)
        torch.cuda.synchronize()
        m = torch.tensor(listed, device="cuda")
        assert torch.equal(g.q[:, m], ref.q[:, m]) and torch.equal(g.nsteps[m], ref.nsteps[m])
        assert torch.equal(g.status[m], ref.status[m]) and torch.equal(g.lam[m], ref.lam[m])
        assert torch.equal(g.q[:, ~m], start.q[:, ~m]) and bool((g.status[~m] == gray2.ACTIVE).all())
        assert bool((g.nsteps[~m] == 0).all()) and gray2.stats_dict(stats)["n_active"] == 500


def test_fma_probes_of_the_bench_run_in_every_form():
    """The FMA-only kernels behind bench.py's fma_probe_* fields live in bench_probe.cu (not in the product
    library): every operand form launches, bad forms are refused."""
    import bench
    lib = bench.load_probe()
    for prec, dtype, forms in ((0, torch.float64, (0, 1, 2)), (1, torch.float32, (0, 1, 2, 3))):
        scratch = torch.zeros(8, dtype=dtype, device="cuda")
        for form in forms:
            assert lib.bench_fma_probe(prec, form, 4, 64, 10, scratch.data_ptr(), None) == 0
    torch.cuda.synchronize()
    assert lib.bench_fma_probe(0, 3, 4, 64, 10, scratch.data_ptr(), None) == 1


def test_backward_direction_and_lambda_clip():
    xu8, _ = inputs.cfg4_ensemble(64)
    g = gray2.init_timelike(0.7, xu8)
    o = oracle.init_timelike(0.7, xu8)
    fwd = sc_pair(mode=0, h_fixed=0.3, max_steps=100000)
    gray2.integrate(g, 100.0, fwd[0])       # 333 full steps + one clipped step of 0.1
    oracle.integrate(o, 100.0, fwd[1])
    gst = to_oracle_state(g)
    assert (gst.nsteps == 334).all() and np.array_equal(gst.nsteps, o.nsteps)
    assert np.max(np.abs(gst.lam - 100.0)) < 1e-12 and (gst.status == gray2.ACTIVE).all()
    assert state_rel_error(gst.q, o.q, 0.7).max() < TOL_STATE_F64
    bwd = sc_pair(mode=0, h_fixed=0.3, dir=-1, max_steps=100000)
    gray2.integrate(g, 0.0, bwd[0])
    back = to_oracle_state(g)
    assert np.max(np.abs(back.lam)) < 1e-12
    assert np.max(np.abs(back.q - xu8.T)) < 1e-6     # retraces the segment to truncation error


@pytest.mark.parametrize("prec", [gray2.F64, gray2.F32], ids=["f64", "f32"])
def test_clipped_step_lands_on_the_end_value_exactly(prec):
    """DESIGN R22 on the GPU, all integrators: after a clipped last step the clock IS lambda_end (t_end), also where
    lambda + (lambda_end - lambda) != lambda_end in double (0.03 -> 0.283 overshoots, 0.05 -> 0.216 falls short), and
    the step counts equal the oracle's; a second identical call does nothing."""
    xu8, _ = inputs.cfg4_ensemble(100)
    for first, second in ((0.03, 0.283), (0.05, 0.216)):
        for name, grun, orun in (("affine", gray2.integrate, oracle.integrate),
                                 ("coordtime", gray2.integrate_coordtime, oracle.integrate_coordtime),
                                 ("diagnostics", lambda *a, **k: gray2.integrate_diagnostics(*a, **k) and k.get("stats"),
                                  lambda *a: oracle.integrate_diagnostics(*a)[0])):
            g = gray2.init_timelike(0.7, xu8, prec=prec)
            o = oracle.init_timelike(0.7, xu8)
            gsc, osc = sc_pair(mode=0, h_fixed=1.0, max_steps=10 ** 6)
            stats = gray2.new_stats()
            for end in (first, second, second):
                grun(g, end, gsc, stats=stats)
                ostats = orun(o, end, osc)
                torch.cuda.synchronize()
                assert gray2.stats_dict(stats) == ostats, (name, end)
                clock = g.q[0].double() if name == "coordtime" else g.lam
                # (the coordinate-time clock is q[0] itself: a float in FP32 states, so the end value as a float)
                expect = float(np.float32(end)) if (name == "coordtime" and prec == gray2.F32) else end
                assert bool((clock == expect).all()), (name, end, clock[:3])
            assert ostats["steps"] == 0 and bool((g.nsteps == 2).all())


# ---- full-size configs, in the launch configuration bench.py times, against sampled oracle rays -----

@pytest.mark.parametrize("cfg,nsample", [(inputs.CFG3_NULL, 1536), (inputs.CFG2_NULL, 1024)], ids=lambda c: getattr(c, "name", str(c)))
def test_full_size_image_sampled_parity(cfg, nsample):
    g0, g, gstats = run_gpu_image(cfg)
    assert gstats["n_active"] == 0 and gstats["n_invalid"] == 0 and gstats["n_maxsteps"] <= 2
    assert gstats["n_captured"] + gstats["n_escaped"] + gstats["n_maxsteps"] == cfg.n
    assert gstats["steps"] == int(g.nsteps.sum(dtype=torch.int64).item())
    rng = np.random.default_rng(1706)
    idx = np.sort(rng.choice(cfg.n, nsample, replace=False))
    full0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o = take(full0, idx)
    oracle.integrate(o, INF, image_sc(cfg)[1])
    gst = take(to_oracle_state(g), idx)
    xi, eta, _, _ = ih.ray_constants(take(full0, idx))
    _, beta = ih.pixel_grid(cfg)
    a_inf, b_inf = ih.asymptotic_image_point(full0.a_eff, cfg.inclination, xi, eta, np.where(beta[idx] >= 0, 1.0, -1.0))
    d = ih.band_distance(cfg.a, cfg.inclination, a_inf, b_inf)
    outside = d > 1e-3
    assert np.array_equal(gst.status[outside], o.status[outside]) and np.array_equal(gst.nsteps[outside], o.nsteps[outside])
    assert state_rel_error(gst.q[:, outside], o.q[:, outside], o.a_eff).max() < TOL_STATE_F64
    # property that holds at any size: the mask equals Carter's potential for every sampled ray outside the band,
    # and the captured fraction of the WHOLE image is the area of Bardeen's curve over the field of view
    mask = ih.potential_mask(full0.a_eff, xi, eta, 900.0)
    assert np.array_equal((gst.status == gray2.CAPTURED)[outside], mask[outside])
    ca, cb = __import__("closed_forms").bardeen_curve(cfg.a, cfg.inclination)
    order = np.argsort(ca)
    area = 2.0 * np.trapezoid(cb[order], ca[order])
    assert abs(gstats["n_captured"] / cfg.n - area / (2 * cfg.fov) ** 2) < 2e-3


@pytest.mark.parametrize("form", ["affine", "coordtime"])
def test_fp32_trace_split_into_calls_stays_within_rounding(form):
    """An FP32 state is plain float at every call boundary (include/gray2.h): the residuals of the compensated sums are
    dropped when a geodesic is stored, so a trace made in several calls differs from the same trace made in one -- by
    one float rounding of the state per call, which the geodesic then carries like a rounding of its input.  Bounded
    here: eight segments against one call, every ray that is not critical for FP32 (the criterion of the parity tests)
    ends with the same status, on the same line of flight: the impact vector x x v_hat, which does not depend on where
    along the ray the two traces stop, agrees to a few float ulp of r."""
    cfg = inputs.CFG3_NULL.scaled(80, 64)
    gsc, _ = image_sc(cfg)
    kw = image_sc_kw(cfg)
    run = gray2.integrate_coordtime if form == "coordtime" else gray2.integrate
    one = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=gray2.F32)
    o0 = to_oracle_state(one)
    many = one.clone()
    run(one, INF, gsc)
    for end in (150.0, 400.0, 700.0, 900.0, 980.0, 1010.0, 1300.0, INF):      # lambda or t: about the same far out
        run(many, end, gsc)
    torch.cuda.synchronize()
    a, b = to_oracle_state(one), to_oracle_state(many)
    sens = twin_sensitivity(o0, kw)
    noncrit = sens <= TOL_STATE_F32
    assert noncrit.mean() > 0.9 and np.array_equal(a.status[noncrit], b.status[noncrit])
    # a call that ends at lambda_end clips its last step, so the split trace has up to seven steps more
    assert (np.abs(a.nsteps - b.nsteps)[noncrit] <= 8).all() and (b.nsteps >= a.nsteps)[noncrit].all()
    near = noncrit & (np.abs(a.nsteps - b.nsteps) <= 8)
    r_a = np.array([oracle.ks_r(a.a_eff, *a.q[1:4, k]) for k in range(a.n)])
    # the two traces stop a few (clipped) steps apart: compare what does not depend on where along the ray they stop
    va, vb = a.q[5:8] / np.linalg.norm(a.q[5:8], axis=0), b.q[5:8] / np.linalg.norm(b.q[5:8], axis=0)
    dv = np.linalg.norm(va - vb, axis=0)          # up to 8 steps further out the ray has bent by up to ~2 b dr / r^2 ~ 1e-5
    bvec_a = np.cross(a.q[1:4].T, va.T)           # impact vector x x v_hat: constant far out
    bvec_b = np.cross(b.q[1:4].T, vb.T)
    db = np.linalg.norm(bvec_a - bvec_b, axis=1) / r_a
    esc = near & (a.status == gray2.ESCAPED)
    print("[fp32 split calls] %s: direction differs by median %.2e max %.2e, impact vector / r by median %.2e max %.2e (%d escaped rays)"
          % (form, np.median(dv[esc]), dv[esc].max(), np.median(db[esc]), db[esc].max(), esc.sum()))
    # measured: impact vector / r median 3e-8, max 1.4e-7 (half a float ulp is 3e-8)
    assert dv[esc].max() < TOL_STATE_F32 and db[esc].max() < 2e-6 and np.median(db[esc]) < 2e-7


def test_full_size_headline_image_fp32_sampled_parity():
    """cfg3 at 1024 x 1024 in FP32 -- the workload and the kernel (packed 256 x 2, the default at this size) of the
    bench line's fp32 block -- against 1,536 sampled oracle rays fed the float initial state: north_star's FP32 clause
    on every non-critical sampled ray.  Also printed: how many of the rays the criterion excludes were within 1e-4
    anyway, so that its slack stays visible."""
    cfg = inputs.CFG3_NULL
    g0, g, gstats = run_gpu_image(cfg, prec=gray2.F32)
    assert gstats["n_active"] == 0 and gstats["n_invalid"] == 0 and gstats["n_maxsteps"] <= 2
    assert gstats["steps"] == int(g.nsteps.sum(dtype=torch.int64).item())
    rng = np.random.default_rng(1706)
    idx = np.sort(rng.choice(cfg.n, 1536, replace=False))
    o0 = take(to_oracle_state(g0), idx)              # the same inputs: the float initial state, widened
    o = o0.copy()
    kw = image_sc_kw(cfg)
    oracle.integrate(o, INF, oracle.step_control(**kw))
    gst = take(to_oracle_state(g), idx)
    sens = twin_sensitivity(o0, kw)
    err = state_rel_error(gst.q, o.q, o.a_eff)
    noncrit, same = assert_fp32_parity(cfg.name + " full size, sampled", gst, o, sens, err, make_straddle_check(o0, gst, o, kw))
    agree = (gst.status == o.status) & (gst.nsteps == o.nsteps)
    fine_anyway = int(((~noncrit) & agree & (err < TOL_STATE_F32)).sum())
    print("[fp32 parity] %s: of the %d sampled rays excluded as critical, %d were within %.0e anyway; beyond it on all rays: %d"
          % (cfg.name, int((~noncrit).sum()), fine_anyway, TOL_STATE_F32, int((~(agree & (err < TOL_STATE_F32))).sum())))
    xi, eta, _, _ = ih.ray_constants(o0)
    mask = ih.potential_mask(o0.a_eff, xi, eta, 900.0)
    assert np.array_equal((gst.status == gray2.CAPTURED)[noncrit], mask[noncrit])
    ca, cb = __import__("closed_forms").bardeen_curve(cfg.a, cfg.inclination)
    order = np.argsort(ca)
    area = 2.0 * np.trapezoid(cb[order], ca[order])
    assert abs(gstats["n_captured"] / cfg.n - area / (2 * cfg.fov) ** 2) < 2e-3


def test_cfg4_ensemble_sample_parity_and_drift():
    xu8, meta = inputs.cfg4_ensemble(4096)
    gsc, osc = sc_pair(mode=0, h_fixed=0.5, max_steps=3000)
    g = gray2.init_timelike(0.7, xu8)
    gi0 = [t.cpu().numpy() for t in gray2.invariants(g)]
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    o = oracle.init_timelike(0.7, xu8)
    oi0 = oracle.invariants(o)
    oracle.integrate(o, INF, osc)
    gst = to_oracle_state(g)
    assert gray2.stats_dict(stats)["steps"] == 4096 * 3000 and (gst.status == gray2.MAXSTEPS).all()
    # 3000 steps ~ several radial periods.  The two sides round in different orders (Christoffel form vs
    # regrouped form); eccentric orbits with a deep periapsis amplify that difference along the orbit (phase
    # error).  Which orbits are critical is decided by the oracle alone (twin orbits displaced by the accumulated
    # rounding of 3000 steps, gpu_helpers.accumulated_rounding_f64); 1e-9 holds on EVERY other one.
    err = state_rel_error(gst.q, o.q, 0.7)
    kw = dict(mode=0, h_fixed=0.5, max_steps=3000)
    sens = twin_sensitivity(oracle.init_timelike(0.7, xu8), kw, rel_delta=accumulated_rounding_f64(3000), twins=TWINS_ORBIT)
    noncrit = sens <= TOL_STATE_F64
    print("[cfg4 sample] %d of 4096 orbits critical; max error on the others %.2e, on all %.2e" % ((~noncrit).sum(), err[noncrit].max(), err.max()))
    assert noncrit.mean() > 0.99 and err[noncrit].max() < TOL_STATE_F64, (noncrit.mean(), err[noncrit].max())
    # and without any criterion: every orbit within 10 x the tolerance (measured 7.4e-10), the criterion excluding
    # no more than a handful (measured 3 of 4096)
    assert err.max() < 10 * TOL_STATE_F64 and (~noncrit).sum() <= 8, (err.max(), (~noncrit).sum())
    gi1 = [t.cpu().numpy() for t in gray2.invariants(g)]
    oi1 = oracle.invariants(o)
    from gpu_helpers import invariant_term_scales
    scales = invariant_term_scales(o.q)
    for k in range(4):
        scale = scales[k]
        assert np.max(np.abs((gi1[k] - gi0[k]) - (oi1[k] - oi0[k])) / scale) < 1e-12


def test_cfg4_full_size_sampled_parity():
    """BASELINE.json configs[3] at full size (1,048,576 particles x 100,000 fixed steps) in the launch
    configuration bench.py uses; 768 sampled particles against the oracle: 512 evenly spaced through the ensemble
    and the 256 with the deepest periapses (smallest r_p = p / (1 + e): the orbits that amplify a rounding-level
    difference between the two formulations most, "u^2 ... increases")."""
    n, nsteps = 1 << 20, 100000
    xu8, meta = inputs.cfg4_ensemble(n)
    gsc, osc = sc_pair(mode=0, h_fixed=0.5, max_steps=nsteps)
    g = gray2.init_timelike(0.7, xu8)
    gi0 = [t.cpu().numpy() for t in gray2.invariants(g)]
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    sd = gray2.stats_dict(stats)
    assert sd["n_invalid"] == 0 and sd["n_active"] == 0 and sd["n_escaped"] == 0
    assert sd["n_maxsteps"] + sd["n_captured"] == n and sd["n_captured"] < 100     # marginal orbits may plunge at h = 0.5
    assert sd["steps"] == int(g.nsteps.sum(dtype=torch.int64).item())
    even = np.arange(0, n, n // 512)[:512]
    rp = meta["p"] / (1.0 + meta["e"])
    deep = np.setdiff1d(np.argsort(rp, kind="stable")[:300], even)[:256]
    idx = np.concatenate([even, deep])
    o = oracle.init_timelike(0.7, xu8[idx])
    oi0 = oracle.invariants(o)
    oracle.integrate(o, INF, osc)
    tidx = torch.tensor(idx, device="cuda")
    assert np.array_equal(g.nsteps[tidx].cpu().numpy(), o.nsteps) and np.array_equal(g.status[tidx].cpu().numpy(), o.status)
    err = state_rel_error(g.q[:, tidx].cpu().numpy(), o.q, 0.7)
    orbiting = o.status == oracle.MAXSTEPS
    print("[cfg4 full size] state error after 1e5 steps: evenly spaced max %.2e; deepest periapses (r_p %.3f..%.3f, %d still "
          "orbiting) median %.2e 99%% %.2e max %.2e" % (err[:512].max(), rp[deep].min(), rp[deep].max(), orbiting[512:].sum(),
                                                         np.median(err[512:][orbiting[512:]]), np.quantile(err[512:][orbiting[512:]], 0.99),
                                                         err[512:][orbiting[512:]].max()))
    # Which of these orbits are critical over 1e5 steps is decided by the oracle alone: twin orbits displaced by the
    # accumulated rounding of the run (gpu_helpers.accumulated_rounding_f64: 2^-52 sqrt(4 nsteps) = 1.4e-13 relative);
    # 1e-9 holds on EVERY orbit whose final state is stable to 1e-9 under that displacement.
    kw = dict(mode=0, h_fixed=0.5, max_steps=nsteps)
    sens = twin_sensitivity(oracle.init_timelike(0.7, xu8[idx]), kw, rel_delta=accumulated_rounding_f64(nsteps), twins=TWINS_ORBIT)
    noncrit = orbiting & (sens <= TOL_STATE_F64)
    print("[cfg4 full size] critical or plunged: %d of the 512 evenly spaced, %d of the 256 deepest; max error on the others %.2e"
          % ((~noncrit[:512]).sum(), (~noncrit[512:]).sum(), err[noncrit].max()))
    assert noncrit[:512].mean() > 0.95 and err[noncrit].max() < TOL_STATE_F64, (noncrit[:512].mean(), err[noncrit].max())
    # Unconditional ceilings beside the criterion, from the recorded run (evenly spaced: max 1.07e-9, 20 of 512 excluded;
    # deepest periapses: max 4.3e-7 over the orbiting ones, 101 of 256 excluded): the criterion may not hide an orbit that
    # is off by more than the phase growth of 1e5 steps explains, nor grow to exclude more than it does today.
    assert err[:512][orbiting[:512]].max() < 1e-8 and err[512:][orbiting[512:]].max() < 5e-6
    assert (~noncrit[:512]).sum() <= 26 and (~noncrit[512:]).sum() <= 115, ((~noncrit[:512]).sum(), (~noncrit[512:]).sum())
    gi1 = [t.cpu().numpy() for t in gray2.invariants(g)]
    oi1 = oracle.invariants(o)
    from gpu_helpers import invariant_term_scales
    scales = invariant_term_scales(o.q)
    names = ("E", "Lz", "Q", "u.u")
    for k in range(4):
        gd, od = (gi1[k] - gi0[k])[idx], oi1[k] - oi0[k]
        sel = orbiting
        # beside the term-scaled bound of DESIGN section 6, the plain figure: the difference of the two drifts
        # relative to the drift itself (rms over the sample) and to the invariant
        print("[cfg4 full size] drift of %-3s: rms %.2e; GPU - oracle: rms %.2e = %.1e of the drift, max %.2e of the invariant's terms"
              % (names[k], np.sqrt(np.mean(od[sel] ** 2)), np.sqrt(np.mean((gd - od)[sel] ** 2)),
                 np.sqrt(np.mean((gd - od)[sel] ** 2)) / max(np.sqrt(np.mean(od[sel] ** 2)), 1e-300),
                 np.max(np.abs(gd - od)[sel] / scales[k][sel])))
        assert np.max(np.abs(gd - od)[:512] / scales[k][:512]) < 1e-12
        assert np.max(np.abs(gd - od)[sel] / scales[k][sel]) < 1e-11
    # drift stays at the RK4 truncation level over 1e5 steps
    alive = g.status.cpu().numpy() == gray2.MAXSTEPS      # the few plunging particles end inside the horizon region
    dE, dn = (gi1[0] - gi0[0])[alive], (gi1[3] - gi0[3])[alive]
    assert np.abs(dE).max() < 1e-2 and np.abs(dn).max() < 1e-2              # worst: deep-periapsis orbits at h = 0.5
    assert np.sqrt(np.mean(dE ** 2)) < 1e-4 and np.sqrt(np.mean(dn ** 2)) < 1e-4


@pytest.mark.parametrize("prec", [gray2.F64, gray2.F32], ids=["f64", "f32"])
def test_cfg5_full_size_sampled_parity(prec):
    """BASELINE.json configs[4]: 4096 x 4096 rays (16.8 M), heavy divergence in path length."""
    cfg = inputs.CFG5_NULL
    gsc, osc = image_sc(cfg)
    g = gray2.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny, prec=prec)
    rng = np.random.default_rng(5)
    idx = np.sort(rng.choice(cfg.n, 768, replace=False))
    tidx = torch.tensor(idx, device="cuda")
    g0q = g.q[:, tidx].double().cpu().numpy()              # the sampled rays' initial state as the kernel reads it
    stats = gray2.new_stats()
    gray2.integrate(g, INF, gsc, stats=stats)
    sd = gray2.stats_dict(stats)
    assert sd["n_active"] == 0 and sd["n_invalid"] == 0 and sd["n_maxsteps"] <= 4
    assert sd["n_captured"] + sd["n_escaped"] + sd["n_maxsteps"] == cfg.n
    assert sd["steps"] == int(g.nsteps.sum(dtype=torch.int64).item())
    ca, cb = __import__("closed_forms").bardeen_curve(cfg.a, cfg.inclination)
    order = np.argsort(ca)
    area = 2.0 * np.trapezoid(cb[order], ca[order])
    assert abs(sd["n_captured"] / cfg.n - area / (2 * cfg.fov) ** 2) < 1e-3
    full0 = oracle.init_null(cfg.a, cfg.r_obs, cfg.inclination, cfg.fov, cfg.fov, cfg.nx, cfg.ny)
    o0 = take(full0, idx)
    del full0
    if prec == gray2.F32:
        o0.q[:] = g0q                                      # the same inputs: the float initial state, widened
    o = o0.copy()
    oracle.integrate(o, INF, osc)
    gq = g.q[:, tidx].double().cpu().numpy()
    gs, gn = g.status[tidx].cpu().numpy(), g.nsteps[tidx].cpu().numpy()
    xi, eta, _, _ = ih.ray_constants(o0)
    alpha, beta = ih.pixel_grid(cfg)
    a_inf, b_inf = ih.asymptotic_image_point(o0.a_eff, cfg.inclination, xi, eta, np.where(beta[idx] >= 0, 1.0, -1.0))
    d = ih.band_distance(cfg.a, cfg.inclination, a_inf, b_inf)
    if prec == gray2.F64:
        outside = d > 1e-3
        assert np.array_equal(gs[outside], o.status[outside]) and np.array_equal(gn[outside], o.nsteps[outside])
        assert state_rel_error(gq[:, outside], o.q[:, outside], o.a_eff).max() < TOL_STATE_F64
    else:
        kw = image_sc_kw(cfg)
        gst = oracle.State(len(idx), gq, g.lam[tidx].cpu().numpy(), gs, gn, o.a_eff, o.kind, o.reversed, o.coords)
        sens = twin_sensitivity(o0, kw)
        assert_fp32_parity(cfg.name + " full size, 768 sampled rays", gst, o, sens, state_rel_error(gq, o.q, o.a_eff),
                           make_straddle_check(o0, gst, o, kw))
