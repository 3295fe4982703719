#!/usr/bin/env python
"""bench.py -- throughput of the vog hot path on B200 (contract: see the task statement / DESIGN.md 9).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--no-sweep] [--no-cpu]

Workload (BASELINE.json metric): one Strang step (x/2 - field - v - x/2, 3 fused advections +
density + Poisson) of the fp32 delta-f scheme on a 2048 x 2048 grid, LAG17, nonlinear-Landau
initial data.  One bench "step" advances a BATCH of independent replicas of that grid by one
Strang step each; the batch (16 x 16 MiB = 256 MiB) is larger than the 126 MB L2, so every
replica is L2-cold when its turn comes again.  value = phase-space cells advanced per second by
the whole job.  Multi-GPU = independent replicas per rank (the path does not shard).

Output (rank 0, stdout): first the detail records -- one JSON line per row of the config-4 sweep
({"sweep_row": ...}), one for the small grids, one for the per-advection oracle timings -- and then, as the
LAST line, the short result record the driver parses (< 2.5 KB).  The detail records are also written to
gpurun_out/bench_detail.json when that directory can be created.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1301_5892_b200 import inputs  # noqa: E402

METRIC = "phase-space cell-updates/s per Strang step (fp32 delta-f, 2048x2048)"
UNIT = "cell-updates/s"
WORKLOAD = "strang_step_deltaf_2048x2048_lag17"
BATCH = 16


def _traffic():
    """(dram bytes per launch of the roofline kernel, source) from the committed ncu capture, else (None, None).
    It is a constant of that capture (ncu cannot run inside a timed bench), named as such in the record."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        src = None
        for line in open(path):
            key, _, val = line.strip().partition(",")
            if key == "source":
                src = val
            if key == "x_kernel_2048_dram_bytes_per_launch":
                return float(val), src
    except Exception:
        pass
    return None, None


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
        except Exception:
            pass
    return 6650.0, "fallback B200_PROFILING.md 6.65 TB/s"


def _r(x, n=4):
    """round to n significant digits (keeps the result line short)"""
    if x is None:
        return None
    return float("%.*g" % (n, x))


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 50 ms DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _oracle_step_rate(orc, cfg, warmup, steps, budget_s, batch=1):
    """cell-updates/s of the oracle's Strang step on cfg: `warmup` untimed steps, then the BEST of up to `steps`
    timings of `batch` consecutive steps inside budget_s seconds (best of 3)."""
    f = inputs.initial_f(cfg).astype(np.float64)
    feq = orc.Feq.make(cfg.feq)
    for _ in range(warmup):
        f, _E = orc.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
    best, n, t_all = None, 0, time.perf_counter()
    while n < steps and (n == 0 or time.perf_counter() - t_all < budget_s):
        t0 = time.perf_counter()
        for _ in range(batch):
            f, _E = orc.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
        dt = (time.perf_counter() - t0) / batch
        best = dt if best is None else min(best, dt)
        n += 1
    return cfg.Nx * cfg.Nv / best, n, time.perf_counter() - t_all


def reference_arm(args, rank):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only; other ranks exit 0)."""
    if rank != 0:
        return
    from oracle import vog_oracle as orc
    orc.build()
    cfg = inputs.metric_config()
    f = inputs.initial_f(cfg).astype(np.float64)
    feq = orc.Feq.make(cfg.feq)
    for _ in range(args.warmup):
        f, _E = orc.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        f, _E = orc.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
    dt = time.perf_counter() - t0
    val = cfg.Nx * cfg.Nv * args.steps / dt
    sample = "full %dx%d Strang step, 1 replica per step (not a batch), double precision, no FFT" % (cfg.Nx, cfg.Nv)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "batch": 1, "Nx": cfg.Nx, "Nv": cfg.Nv},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="vog")
    ap.add_argument("--no-sweep", action="store_true", help="skip the config-4 advection sweep")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg and the oracle timings of the sweep")
    ap.add_argument("--no-extras", action="store_true", help="skip the concurrent / merged / small-grid variants")
    ap.add_argument("--sweep-only", action="store_true", help="only the config-4 advection sweep (for profiling)")
    ap.add_argument("--sizes", default="512,2048,8192,16384", help="sweep grid sizes N (Nx=Nv=N), BASELINE.json config 4")
    ap.add_argument("--kinds", default="lag3,lag9,lag17,spline", help="sweep interpolators: lagN or spline")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        reference_arm(args, rank)
        return

    import torch
    from paper_1301_5892_b200 import multi, vog

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        multi.init("nccl", device_id=torch.device("cuda", local))
    vog.lib()

    detail = []

    def emit(rec):
        detail.append(rec)
        if rank == 0:
            print(json.dumps(rec), flush=True)

    sizes = tuple(int(x) for x in args.sizes.split(","))
    kinds = tuple((1, 3) if k == "spline" else (0, int(k[3:])) for k in args.kinds.split(","))
    stream = torch.cuda.Stream()
    peak, peak_src = _peaks()
    if args.sweep_only:
        sweep(torch, vog, stream, peak, sizes, kinds, emit, with_oracle=False)
        return
    cfg = inputs.metric_config()
    cells = cfg.Nx * cfg.Nv
    plan = vog.Plan.from_config(cfg, stream=stream)
    f0 = torch.from_numpy(inputs.initial_f(cfg))
    with torch.cuda.stream(stream):
        batch = [f0.cuda(non_blocking=False).clone() for _ in range(BATCH)]
    stream.synchronize()

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            multi.barrier()
            torch.cuda.synchronize()

    def bench_step():
        for fb in batch:
            plan.step(fb, cfg.dt)

    for _ in range(args.warmup):
        bench_step()
    sync_all()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    n0 = plan.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        bench_step()
    ev1.record(stream)
    sync_all()
    ms = ev0.elapsed_time(ev1)
    launches = plan.launch_count() - n0
    clocks = sampler.stop() if rank == 0 else None
    ms = multi.max_over_ranks(ms, device="cuda")
    value = multi.aggregate_throughput(BATCH * cells * args.steps, world, ms)

    # ---- per-kernel timing of the same step on the same stream (roofline of the dominant kernel).  Each call type
    # is enqueued back to back on all replicas of the batch between two events (no host synchronisation inside), so
    # the figure is the average duration in steady state, every replica L2-cold on entry.
    Ed = torch.empty(cfg.Nx, device="cuda", dtype=torch.float32)
    plan.field(batch[0], Ed)

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        tot = 0.0
        reps = min(max(args.steps // 4, 3), 10)
        for _ in range(reps):
            e0.record(stream)
            for fb in batch:
                fn(fb)
            e1.record(stream)
            stream.synchronize()
            tot += e0.elapsed_time(e1)
        return tot / (reps * BATCH)

    with torch.cuda.stream(stream):
        ms_x = timed(lambda fb: plan.advect_x(fb, 0.5 * cfg.dt))      # tables cached: the x kernel alone
        ms_f = timed(lambda fb: plan.field(fb, Ed))                   # density + Poisson
        ms_v = timed(lambda fb: plan.advect_v(fb, Ed, cfg.dt))        # table setup + v kernel (+ delta-f source)
    alg_bytes = 8.0 * cells                      # one read + one write of f per advection
    ach = alg_bytes / (ms_x * 1e-3) / 1e9
    traffic, traffic_src = _traffic()
    roofline = {"bound": "hbm", "kernel": "x-advection kernel, 2048-cell lines (2 of 3 advections)",
                "achieved": _r(ach, 5), "peak": peak, "unit": "GB/s", "frac": _r(ach / peak), "traffic": traffic,
                "traffic_source": traffic_src, "peak_source": peak_src, "alg_bytes_per_launch": alg_bytes,
                "us_per_launch": _r(1e3 * ms_x), "us_v_call": _r(1e3 * ms_v), "us_field": _r(1e3 * ms_f),
                "note": "16 MiB replica: L2-cold on entry, writes stay in L2; HBM-resident sizes: target_8192"}

    extras = {}
    if not args.no_extras:
        # ---- the same batch with the replicas spread over 4 plans on 4 streams (independent problems overlap)
        NS = 4
        streams = [torch.cuda.Stream() for _ in range(NS)]
        plans = [vog.Plan.from_config(cfg, stream=st) for st in streams]
        main_st = torch.cuda.current_stream()

        def conc_step():
            for i, fb in enumerate(batch):
                plans[i % NS].step(fb, cfg.dt)

        for _ in range(args.warmup):
            conc_step()
        sync_all()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(main_st)
        for st in streams:
            st.wait_event(c0)
        for _ in range(args.steps):
            conc_step()
        for st in streams:
            e = torch.cuda.Event()
            e.record(st)
            main_st.wait_event(e)
        c1.record(main_st)
        sync_all()
        cms = multi.max_over_ranks(c0.elapsed_time(c1), device="cuda")
        extras["concurrent_4_streams"] = _r(multi.aggregate_throughput(BATCH * cells * args.steps, world, cms))
        for pl in plans:
            pl.destroy()

        # ---- merged half steps: vog_run(merge=1), 2 advections per step.
        # A different sequence, so it is reported beside `value`, never as `value`.
        MR = 10
        for fb in batch[:2]:
            plan.run(fb, cfg.dt, MR, None, True)
        sync_all()
        m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        mrep = max(1, args.steps // MR)
        m0.record(stream)
        for _ in range(mrep):
            for fb in batch:
                plan.run(fb, cfg.dt, MR, None, True)
        m1.record(stream)
        sync_all()
        mms = multi.max_over_ranks(m0.elapsed_time(m1), device="cuda")
        extras["merged_half_steps"] = _r(multi.aggregate_throughput(BATCH * cells * MR * mrep, world, mms))

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    fh = f0.clone().pin_memory()
    Eh = torch.empty(cfg.Nx, dtype=torch.float32).pin_memory()
    for _ in range(3):
        plan.run_host(fh, cfg.dt, 1, None, Eh)
    sync_all()
    e2e_steps = max(5, min(args.steps, 20))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        plan.run_host(fh, cfg.dt, 1, None, Eh)      # synchronises before returning
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = multi.max_over_ranks(e2e_s, device="cuda")
    serial_value = world * cells * e2e_steps / e2e_s
    # the same per-step traffic with three replicas in flight: vog_run_host_async on three plans / streams, so that one
    # replica's copy in, another's step and a third's copy out overlap (PCIe is full duplex); every step still
    # copies its 16 MiB in from pinned memory and its f and E back out, all inside the timed region
    NP = 3
    pstreams = [torch.cuda.Stream() for _ in range(NP)]
    pplans = [vog.Plan.from_config(cfg, stream=st) for st in pstreams]
    fhs = [f0.clone().pin_memory() for _ in range(NP)]
    Ehs = [torch.empty(cfg.Nx, dtype=torch.float32).pin_memory() for _ in range(NP)]
    for i in range(2 * NP):
        pplans[i % NP].run_host_async(fhs[i % NP], cfg.dt, 1, None, Ehs[i % NP])
    sync_all()
    p_steps = NP * e2e_steps
    t0 = time.perf_counter()
    for i in range(p_steps):
        pplans[i % NP].run_host_async(fhs[i % NP], cfg.dt, 1, None, Ehs[i % NP])
    torch.cuda.synchronize()
    p_s = time.perf_counter() - t0
    p_s = multi.max_over_ranks(p_s, device="cuda")
    for pl in pplans:
        pl.destroy()
    e2e = {"value": _r(world * cells * p_steps / p_s, 5), "unit": UNIT, "h2d_bytes_per_step": 4 * cells,
           "d2h_bytes_per_step": 4 * cells + 4 * cfg.Nx, "steps": p_steps, "replicas_in_flight": NP,
           "serial_value": _r(serial_value, 5),
           "note": "vog_run_host_async, 3 plans/streams: pinned f in, 1 step, f and E out, every step; "
                   "serial_value: vog_run_host"}
    plan.destroy()

    # ---- small grids (configs 0-1: launch/latency-bound: report steps/s)
    if not args.no_extras:
        extras["small_grids_steps_per_s"] = small_grids(torch, vog, stream, emit)

    out = {
        "metric": METRIC, "value": _r(value, 6), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": _r(ms / args.steps, 6), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "Nx": cfg.Nx, "Nv": cfg.Nv, "batch": BATCH, "split": "x/2-field-v-x/2",
                   "interp": "LAG17", "parallelism": "replicas x%d" % world,
                   "l2": "inputs larger than L2: %d replicas = %d MiB, round-robin" % (BATCH, BATCH * 4 * cells >> 20)},
        "gpu_launches": launches, "us_per_replica_step": _r(1e3 * ms / (args.steps * BATCH)),
        "MA_paper_unit": _r(3.0 * value / 1e6), "e2e": e2e, "roofline": roofline,
    }
    out.update(extras)
    if rank == 0:
        out["clocks"] = clocks

    # ---- config-4 sweep (one x- and one v-advection on 512..16384 squared, LAG3/9/17 + spline), detail lines
    if rank == 0 and not args.no_sweep:
        rows = sweep(torch, vog, stream, peak, sizes, kinds, emit, with_oracle=(world == 1 and not args.no_cpu))
        tgt = {}
        for N in (8192, 16384):
            for r in rows:
                if r["N"] == N and r["kind"] == "lagrange" and r["order"] == 17:
                    tgt[str(N)] = {"x_kernel_frac": _r(r["x_kernel_only"]["frac_hbm"]),
                                   "x_call_frac": _r(r["x"]["frac_hbm"]), "v_call_frac": _r(r["v"]["frac_hbm"]),
                                   "v_out_of_place_frac": _r(r.get("v_out_of_place", {}).get("frac_hbm")),
                                   "step_frac_28B": _r(r["strang_step"]["frac_hbm"]),
                                   "direct_stencil_x_v_step": [_r(r.get("direct_stencil", {}).get(k, {}).get("frac_hbm"))
                                                               for k in ("x_kernel_only", "v_out_of_place", "strang_step")],
                                   "f64_mode_x_step": [_r(r.get("f64_mode", {}).get(k, {}).get("frac_hbm"))
                                                       for k in ("x_kernel_only", "strang_step")]}
        roofline["target_8192"] = tgt.get("8192")
        roofline["at_16384"] = tgt.get("16384")
    # ---- oracle on the host cores (rank 0, N=1 only)
    if rank == 0 and world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(cfg)
    if rank == 0:
        try:
            os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
            with open(os.path.join(ROOT, "gpurun_out", "bench_detail.json"), "w") as fh_:
                json.dump({"result": out, "detail": detail}, fh_, indent=1)
        except Exception:
            pass
        print(json.dumps(out), flush=True)
    if world > 1:
        multi.finalize()


def small_grids(torch, vog, stream, emit):
    """Configs 0 and 1 (64^2 full-f, 256^2 delta-f): Strang steps per second through vog_run (one host call for the
    whole run, energies on the device), the configs' own step counts; first as the launch-per-kernel loop, then as ONE
    persistent cluster kernel for the whole run (vog_plan_tune(29, 1), csrc/vog_small.cu).  The result record holds
    [loop, one kernel] per config."""
    res = {}
    for idx in (0, 1):
        cfg = inputs.config(idx)
        f0 = torch.from_numpy(inputs.initial_f(cfg)).cuda()
        en = torch.empty(cfg.steps, device="cuda", dtype=torch.float64)
        for one_kernel in (0, 1):
            plan = vog.Plan.from_config(cfg, stream=stream)
            if one_kernel:
                plan.tune(29, 1)
            best = None
            for rep in range(4):
                f = f0.clone()
                stream.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                plan.run(f, cfg.dt, cfg.steps, None, False, en)
                e1.record(stream)
                stream.synchronize()
                t = e0.elapsed_time(e1)
                if rep > 0:
                    best = t if best is None else min(best, t)
            plan.destroy()
            name = cfg.name + ("_one_kernel" if one_kernel else "")
            res.setdefault(cfg.name, []).append(_r(cfg.steps / (best * 1e-3)))   # [launch-per-kernel loop, one kernel]
            emit({"small_grid": name, "steps": cfg.steps, "ms_run": best, "steps_per_s": cfg.steps / (best * 1e-3),
                  "us_per_step": 1e3 * best / cfg.steps})
    return res


def _time_calls(torch, stream, fn, warm, reps, inner=1):
    """Median and best, in ms per call, of `reps` timed regions of `inner` back-to-back calls each."""
    for _ in range(warm):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    times = []
    for _ in range(reps):
        e0.record(stream)
        for _ in range(inner):
            fn()
        e1.record(stream)
        stream.synchronize()
        times.append(e0.elapsed_time(e1) / inner)
    return float(np.median(times)), min(times)


def _time_kernel(torch, stream, fn, rec):
    """A kernel-only row: the average launch duration over a timed region of 4 back-to-back launches (what a step
    sees: the launches are chained by programmatic dependent launch), and beside it the event-to-event time of a
    single launch (which includes the launch latency and the ramp of an idle GPU)."""
    r = rec(*_time_calls(torch, stream, fn, 3, 10, inner=4))
    r["us_single_launch"] = 1e3 * _time_calls(torch, stream, fn, 1, 10)[0]
    return r


def sweep(torch, vog, stream, peak, sizes, kinds, emit, with_oracle):
    """BASELINE.json config 4: one x- and one v-advection on N x N, f ~ U[0,1), per-line shifts ~ U[-8,8] cells.
    x / v = the public in-place calls vog_shift_x / vog_shift_v (table setup + kernel), one call per timed region;
    x_kernel_only = vog_advect_x with cached tables and v_out_of_place = vog_shift_v_to: average launch duration over
    timed regions of 4 back-to-back launches (us_single_launch beside it); strang_step = vog_step (28 B/cell: 3
    advections + density), one step per timed region.
    With with_oracle, the oracle's shift_x / shift_v (double, stencil or cyclic solve, all host cores) is timed on the
    same shape next to it for N <= 8192 (best of 3)."""
    orc = None
    if with_oracle:
        from oracle import vog_oracle as orc
        orc.build()
    res = []
    for N in sizes:
        f = torch.rand((N, N), device="cuda", dtype=torch.float32)
        bx = torch.from_numpy(inputs.uniform_shifts(N, 41)).cuda()
        fo = bo = None
        if orc is not None and N <= 8192:
            fo = inputs.uniform_grid(N, N).astype(np.float64)
            bo = inputs.uniform_shifts(N, 41)
        for kind, order in kinds:
            plan = vog.Plan(N, N, 1.0, -1.0, 1.0, kind, order, stream=stream)
            row = {"N": N, "kind": "lagrange" if kind == 0 else "bspline", "order": order}

            def rec(med, best, nbytes=8.0):
                gbs = nbytes * N * N / (med * 1e-3) / 1e9
                return {"us_median": 1e3 * med, "us_best": 1e3 * best, "GBps": gbs, "frac_hbm": gbs / peak,
                        "frac_8TBps": gbs / 8000.0}

            # (public calls and kernel-only rows are timed the same way: 4 back to back per timed region, and the
            # event-to-event time of one isolated call beside it)
            row["x"] = _time_kernel(torch, stream, lambda: plan.shift_x(f, bx), rec)
            row["v"] = _time_kernel(torch, stream, lambda: plan.shift_v(f, bx), rec)
            row["x_kernel_only"] = _time_kernel(torch, stream, lambda: plan.advect_x(f, 0.01), rec)
            if N * N * 4 * 3 < 160e9:
                g = torch.empty_like(f)
                row["v_out_of_place"] = _time_kernel(torch, stream, lambda: plan.shift_v_to(f, g, bx), rec)
                del g
            row["strang_step"] = rec(*_time_calls(torch, stream, lambda: plan.step(f, 1e-3), 2, 5), 28.0)
            row["strang_step"]["cell_updates_per_s"] = N * N / (row["strang_step"]["us_median"] * 1e-6)
            plan.destroy()
            if N >= 1024:
                # the same matrix applied directly (vog_plan_tune(27, 1)): beside the Fourier path,
                # never instead of it -- the north-star fractions above are the Fourier kernels'
                plan = vog.Plan(N, N, 1.0, -1.0, 1.0, kind, order, stream=stream)
                plan.tune(27, 1)
                st = {"x_kernel_only": _time_kernel(torch, stream, lambda: plan.advect_x(f, 0.01), rec)}
                if N * N * 4 * 3 < 160e9:
                    g = torch.empty_like(f)
                    st["v_out_of_place"] = _time_kernel(torch, stream, lambda: plan.shift_v_to(f, g, bx), rec)
                    del g
                st["strang_step"] = rec(*_time_calls(torch, stream, lambda: plan.step(f, 1e-3), 2, 5), 28.0)
                row["direct_stencil"] = st
                plan.destroy()
            if N >= 1024 and N * N * 8 * 3 < 160e9:
                # double-precision mode (vog_*_f64): 16 B per cell and advection, 56 B per cell and
                # Strang step (3 advections + the density read)
                plan = vog.Plan(N, N, 1.0, -1.0, 1.0, kind, order, stream=stream)
                f64 = f.double()
                d = {"x_kernel_only": _time_kernel(torch, stream, lambda: plan.advect_x_f64(f64, 0.01),
                                                   lambda m, b: rec(m, b, 16.0))}
                d["strang_step"] = rec(*_time_calls(torch, stream, lambda: plan.step_f64(f64, 1e-3), 2, 5), 56.0)
                row["f64_mode"] = d
                plan.destroy()
                del f64
            if fo is not None:
                ot = {}
                for name, fn in (("x", orc.shift_x), ("v", orc.shift_v)):
                    best = None
                    for _ in range(3):
                        t0 = time.perf_counter()
                        fn(fo, bo, kind, order)
                        dt = time.perf_counter() - t0
                        best = dt if best is None else min(best, dt)
                    ot[name] = {"s_best_of_3": best, "cell_updates_per_s": N * N / best}
                ot["cores"] = orc.num_threads()
                ot["gpu_over_oracle_x"] = (N * N / (row["x"]["us_median"] * 1e-6)) / ot["x"]["cell_updates_per_s"]
                ot["gpu_over_oracle_v"] = (N * N / (row["v"]["us_median"] * 1e-6)) / ot["v"]["cell_updates_per_s"]
                row["oracle"] = ot
            res.append(row)
            emit({"sweep_row": row})
        del f
    return res


def cpu_baseline(cfg):
    """The oracle's Strang step on the metric grid, host cores: 1 warm-up step, then the best of 3 runs of 40 steps
    (best of 3; about 10 s of oracle work)."""
    from oracle import vog_oracle as orc
    orc.build()
    val, n, secs = _oracle_step_rate(orc, cfg, 1, 3, 25.0, batch=40)
    return {"value": _r(val, 5), "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
            "sample": "best of %d runs of 40 %dx%d Strang steps, 1 warm-up (%.1f s of oracle work; fp64)"
                      % (n, cfg.Nx, cfg.Nv, secs)}


if __name__ == "__main__":
    main()
