#!/usr/bin/env python
"""bench.py -- throughput of the vog hot path on B200 (contract: see the task statement / DESIGN.md).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--no-sweep]

Workload (BASELINE.json metric): one Strang step (x/2 - field - v - x/2, 3 fused advections +
density + Poisson) of the fp32 delta-f scheme on a 2048 x 2048 grid, LAG17, nonlinear-Landau
initial data.  One bench "step" advances a BATCH of independent replicas of that grid by one
Strang step each; the batch (16 x 16 MiB = 256 MiB) is larger than the 126 MB L2, so every
replica is L2-cold when its turn comes again.  value = phase-space cells advanced per second by
the whole job.  Multi-GPU = independent replicas per rank (the path does not shard).
Prints ONE JSON line on rank 0.
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
BATCH = 16


def _traffic():
    """dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/), else None."""
    path = os.path.join(ROOT, "profiles", "r1_traffic.csv")
    try:
        for line in open(path):
            key, _, val = line.strip().partition(",")
            if key == "x_kernel_bench_dram_bytes_per_launch":
                return float(val)
    except Exception:
        pass
    return None


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


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


def reference_arm(args, rank):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
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
        "config": {"workload": "strang_step_deltaf_2048x2048_lag17", "batch": 1, "Nx": cfg.Nx, "Nv": cfg.Nv},
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
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-concurrent", action="store_true", help="skip the 4-stream variant of the timed batch")
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

    sizes = tuple(int(x) for x in args.sizes.split(","))
    kinds = tuple((1, 3) if k == "spline" else (0, int(k[3:])) for k in args.kinds.split(","))
    stream = torch.cuda.Stream()
    if args.sweep_only:
        print(json.dumps({"sweep": sweep(torch, vog, stream, _peaks()[0], sizes, kinds)}))
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

    # ---- the same batch with the replicas spread over 4 plans on 4 streams (independent problems overlap: the
    # single-CTA Poisson solve and the tails of one replica's kernels run under another replica's advections).
    # Reported next to `value`, which stays the one-stream figure.
    concurrent = None
    if not args.no_concurrent:
        NS = 4
        streams = [torch.cuda.Stream() for _ in range(NS)]
        plans = [vog.Plan.from_config(cfg, stream=st) for st in streams]
        main = torch.cuda.current_stream()

        def conc_step():
            for i, fb in enumerate(batch):
                plans[i % NS].step(fb, cfg.dt)

        for _ in range(args.warmup):
            conc_step()
        sync_all()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(main)
        for st in streams:
            st.wait_event(c0)
        for _ in range(args.steps):
            conc_step()
        for st in streams:
            e = torch.cuda.Event()
            e.record(st)
            main.wait_event(e)
        c1.record(main)
        sync_all()
        cms = multi.max_over_ranks(c0.elapsed_time(c1), device="cuda")
        concurrent = {"streams": NS, "value": multi.aggregate_throughput(BATCH * cells * args.steps, world, cms),
                      "unit": UNIT, "ms_per_step": cms / args.steps,
                      "note": "same batch and steps, replicas round-robin over 4 plans/streams"}
        for pl in plans:
            pl.destroy()

    # ---- merged half steps: vog_run(merge=1) takes the two x half steps that
    # meet between consecutive steps as one advection, 2 advections per step instead of 3.  A different (the
    # paper's "vlaso") sequence, so it is reported beside `value`, never as `value`.
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
    merged = {"value": multi.aggregate_throughput(BATCH * cells * MR * mrep, world, mms), "unit": UNIT,
              "us_per_replica_step": 1e3 * mms / (BATCH * MR * mrep),
              "note": "vog_run(merge=1), %d steps per call per replica: x(dt/2) [field v(dt) x(dt)]^(n-1) field v(dt) x(dt/2)" % MR}

    # ---- per-kernel timing of the same step on the same stream (roofline of the dominant kernel)
    # Each kernel type is launched back to back on all replicas of the batch between two events (no host
    # synchronisation inside), so the figure is the average launch duration in steady state.
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
        ms_x = timed(lambda fb: plan.advect_x(fb, 0.5 * cfg.dt))
        ms_f = timed(lambda fb: plan.field(fb, Ed))
        ms_v = timed(lambda fb: plan.advect_v(fb, Ed, cfg.dt))
    peak, peak_src = _peaks()
    alg_bytes = 8.0 * cells                      # one read + one write of f per advection
    ach = alg_bytes / (ms_x * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "osx5_kernel (overlap-save x-advection, block pairs, warp-private; 2048-cell lines)", "achieved": ach, "peak": peak,
                "unit": "GB/s", "frac": ach / peak, "traffic": _traffic(), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes, "ms_per_launch": ms_x,
                "other_kernels_ms": {"advect_v(+delta-f source)": ms_v, "density+poisson": ms_f},
                "note": "2048^2 replica is L2-cold on entry (batch 256 MiB > L2) but 16 MiB fits L2 within a step; "
                        "advect_v here is the standalone in-place call (table setup + kernel + copy back from the "
                        "plan's second grid); inside vog_step the v kernel writes the second grid and the next "
                        "x-advection reads it, so no copy is made; HBM-roofline fractions at 8192^2/16384^2 are in sweep"}

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
    e2e = {"value": world * cells * p_steps / p_s, "unit": UNIT, "h2d_bytes_per_step": 4 * cells,
           "d2h_bytes_per_step": 4 * cells + 4 * cfg.Nx, "steps": p_steps, "replicas_in_flight": NP,
           "serial_value": serial_value,
           "note": "vog_run_host_async on 3 plans/streams round-robin: pinned host f -> device, 1 Strang step, f and E "
                   "back to host, per step; serial_value = the same with one replica at a time (vog_run_host, "
                   "synchronising after every step)"}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "strang_step_deltaf_2048x2048_lag17", "Nx": cfg.Nx, "Nv": cfg.Nv, "batch": BATCH,
                   "split": "x/2-field-v-x/2", "interp": "LAG17", "parallelism": "replicas x%d" % world,
                   "l2": "inputs larger than L2: batch of %d replicas = %d MiB, visited round-robin" % (BATCH, BATCH * 4 * cells >> 20)},
        "gpu_launches": launches, "e2e": e2e, "roofline": roofline, "concurrent": concurrent, "merged": merged,
        "MA_paper_unit": 3.0 * value / 1e6,
    }
    if rank == 0:
        out["clocks"] = clocks

    # ---- config-4 sweep at the north-star size (8192^2), one x- and one v-advection
    if rank == 0 and not args.no_sweep:
        out["sweep"] = sweep(torch, vog, stream, peak, sizes, kinds)
    # ---- oracle on the host cores (rank 0, N=1 only)
    if rank == 0 and world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(cfg)
    plan.destroy()
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        multi.finalize()


def sweep(torch, vog, stream, peak, sizes=(2048, 8192), kinds=((0, 17), (0, 3), (1, 3))):
    res = []
    for N in sizes:
        f = torch.rand((N, N), device="cuda", dtype=torch.float32)
        bx = torch.from_numpy(inputs.uniform_shifts(N, 41)).cuda()
        for kind, order in kinds:
            plan = vog.Plan(N, N, 1.0, -1.0, 1.0, kind, order, stream=stream)
            row = {"N": N, "kind": "lagrange" if kind == 0 else "bspline", "order": order}
            for name, fn in (("x", plan.shift_x), ("v", plan.shift_v)):
                for _ in range(3):
                    fn(f, bx)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                times = []
                for _ in range(10):
                    e0.record(stream); fn(f, bx); e1.record(stream)
                    stream.synchronize()
                    times.append(e0.elapsed_time(e1))
                med = float(np.median(times))
                gbs = 8.0 * N * N / (med * 1e-3) / 1e9
                row[name] = {"ms_median": med, "ms_best": min(times), "GBps": gbs, "frac_hbm_measured": gbs / peak,
                             "frac_hbm_8TBps": gbs / 8000.0}
            row["note"] = "vog_shift_x/v calls: table setup + kernel (+ copy back for v, whose kernel is out of place)"
            # the x kernel alone (vog_advect_x caches its tables per dt) and a whole Strang step (in which the
            # v kernel writes the plan's second grid and no copy is made), on the same grid
            for _ in range(3):
                plan.advect_x(f, 0.01)
            times = []
            for _ in range(10):
                e0.record(stream); plan.advect_x(f, 0.01); e1.record(stream)
                stream.synchronize()
                times.append(e0.elapsed_time(e1))
            med = float(np.median(times))
            gbs = 8.0 * N * N / (med * 1e-3) / 1e9
            row["x_kernel_only"] = {"ms_median": med, "GBps": gbs, "frac_hbm_measured": gbs / peak}
            # the v kernel out of place (table setup + kernel, no copy back): what vog_step runs
            if N * N * 4 * 3 < 160e9:
                g = torch.empty_like(f)
                for _ in range(3):
                    plan.shift_v_to(f, g, bx)
                times = []
                for _ in range(10):
                    e0.record(stream); plan.shift_v_to(f, g, bx); e1.record(stream)
                    stream.synchronize()
                    times.append(e0.elapsed_time(e1))
                med = float(np.median(times))
                gbs = 8.0 * N * N / (med * 1e-3) / 1e9
                row["v_out_of_place"] = {"ms_median": med, "GBps": gbs, "frac_hbm_measured": gbs / peak,
                                         "note": "vog_shift_v_to: table setup + kernel, src -> dst"}
                if N >= 1024:
                    # control: the loads and stores of the x kernel without the transform (memory-system floor)
                    for _ in range(3):
                        plan.probe_x_memory_pattern(f, g)
                    times = []
                    for _ in range(10):
                        e0.record(stream); plan.probe_x_memory_pattern(f, g); e1.record(stream)
                        stream.synchronize()
                        times.append(e0.elapsed_time(e1))
                    med = float(np.median(times))
                    gbs = 8.0 * N * N / (med * 1e-3) / 1e9
                    row["x_memory_pattern"] = {"ms_median": med, "GBps": gbs, "frac_hbm_measured": gbs / peak,
                                               "note": "vog_probe_x_memory_pattern: the x kernel's loads and stores, no transform"}
                del g
            for _ in range(2):
                plan.step(f, 1e-3)
            times = []
            for _ in range(5):
                e0.record(stream); plan.step(f, 1e-3); e1.record(stream)
                stream.synchronize()
                times.append(e0.elapsed_time(e1))
            med = float(np.median(times))
            gbs = 28.0 * N * N / (med * 1e-3) / 1e9     # 3 advections x 8 B + 4 B density read per cell
            row["strang_step"] = {"ms_median": med, "cell_updates_per_s": N * N / (med * 1e-3), "GBps_28B_per_cell": gbs,
                                  "frac_hbm_measured": gbs / peak}
            res.append(row)
            plan.destroy()
        del f
    return res


def cpu_baseline(cfg):
    from oracle import vog_oracle as orc
    orc.build()
    f = inputs.initial_f(cfg).astype(np.float64)
    feq = orc.Feq.make(cfg.feq)
    t0 = time.perf_counter()
    n = 0
    while n < 3 and time.perf_counter() - t0 < 20.0:
        f, _E = orc.step(f, cfg.L, cfg.vmin, cfg.vmax, cfg.dt, cfg.kind, cfg.order, feq, cfg.split)
        n += 1
    dt = time.perf_counter() - t0
    return {"value": cfg.Nx * cfg.Nv * n / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
            "sample": "%d full %dx%d Strang steps of one replica (double precision, direct stencils, naive-DFT field)"
                      % (n, cfg.Nx, cfg.Nv)}


if __name__ == "__main__":
    main()
