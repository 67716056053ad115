#!/usr/bin/env python
"""bench.py — Teukolsky grid-point updates/s on B200 (BASELINE.json metric).

A "step" is one full Lax-Wendroff iteration (half step + full step + boundary/polar conditions + observer
sample) over the whole grid.  Default workload at N = 1: BASELINE.json configs[1]
(Kerr a=0.9, s=-2, m=2, fp64, 16384 x 64), with dd (configs[2]) and qd (configs[3]) reported beside it in
`per_precision`.  One JSON line on stdout (rank 0).  See DESIGN.md §7 for every field.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--precision 1|2|4] [--workload cfg2|cfg3|cfg4|sweep:NRxNT]
  python bench.py --impl reference ...     # the oracle on the host cores (same metric, bounded sample)
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

ALG_BYTES_PER_UPDATE = {1: 192.0, 2: 384.0, 4: 768.0}     # 4L read + 4L write + 16L coefficients, x 8 B
FALLBACK_HBM_GBS = 6650.0
FP64_INST_PER_UPDATE = {2: 1294.0, 4: 13320.0}            # DADD + DMUL + DFMA thread instructions per update, ncu (profiles/)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=200)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--no-extra", action="store_true", help="skip the dd/qd side measurements and the cpu baseline")
    ap.add_argument("--option", action="append", default=[], help="key=value passed to teuk_set_option")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "slabs"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE problem cut into r* slabs with a halo "
                         "exchange per 32 iterations (NEXT-4, strong scaling; paper_1006_0663_b200/slabs.py)")
    ap.add_argument("--precisions", default="", help="--sweep: comma-separated limb counts to run (default 1,2,4)")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json config 5: one JSON line per (N_r, N_theta, precision) cell")
    return ap.parse_args()


def workload(name: str):
    from paper_1006_0663_b200 import inputs
    if name.startswith("cfg"):
        return inputs.config(int(name[3:]))
    if name.startswith("sweep:"):
        dims, _, prec = name[6:].partition(":")
        nr, nt = dims.lower().split("x")
        return inputs.sweep_cell(int(nr), int(nt), int(prec or 1))
    raise SystemExit(f"unknown workload {name}")


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._pump, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for n, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; each step a bounded sample (a radial
    window of the workload's grid, same dr*, dtheta, dt, coefficients)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle
    from paper_1006_0663_b200 import inputs
    import numpy as np
    w = workload(args.workload)
    n_win = min(w.n_r, 2048)
    i_lo = max(0, int((inputs.pulse_parameters(w)[0] - w.rstar_min) / w.dr) - n_win // 2)
    cores = oracle.set_threads(0)
    o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win)
    u0 = inputs.initial_state(w)[..., i_lo:i_lo + n_win]
    o.set_initial(np.ascontiguousarray(u0))
    per = {1: 1, 2: 1, 4: 1}[w.precision]
    o.step(args.warmup * per if w.precision == 1 else min(args.warmup, 2))
    steps = args.steps if w.precision == 1 else max(1, min(args.steps, 20))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    val = n_win * w.n_theta * steps / dt
    sample = f"radial window of {n_win} of {w.n_r} columns x {w.n_theta} rows, {steps} steps"
    line = {"impl": "reference", "metric": "Teukolsky grid-point updates/s", "value": val, "unit": "updates/s",
            "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {1: "f64", 2: "f64x2 (double-double)", 4: "f64x4 (quad-double)"}[w.precision],
            "data": "synthetic", "config": {"workload": w.name, "n_r": w.n_r, "n_theta": w.n_theta, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "updates/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def make_solver(teuk, w, options, obs_capacity):
    g = teuk.Teuk.from_workload(w, obs_capacity=obs_capacity)
    for kv in options:
        k, _, v = kv.partition("=")
        g.set_option(k, float(v))
    ro, to = w.observer
    g.set_observer(ro, to, obs_capacity)
    return g


def time_device(torch, teuk, w, steps, warmup, options, dist=None):
    """inputs resident in HBM; CUDA events on the stream the kernels are launched on."""
    from paper_1006_0663_b200 import inputs
    g = make_solver(teuk, w, options, warmup + steps)
    u0 = torch.from_numpy(inputs.initial_state(w)).to(g.device)
    g.set_initial(u0)
    g.step(warmup)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    n0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    g.step(steps)
    e1.record(g.stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    if dist is not None:
        dist.barrier()
    launches = g.launch_count() - n0
    geom = g.step_geometry()
    ser = g.observe(4, allow_nonfinite=True)
    finite = bool(torch.isfinite(g.read_device()).all().item()) and g.last_observe_status == 0
    g.close()
    return ms, launches, geom, finite


def time_e2e(torch, teuk, w, steps, options):
    """same job through the C ABI with HOST buffers: teuk_set_initial (H2D from pinned memory) + teuk_step +
    teuk_read (D2H into pinned memory) all inside the timed region."""
    from paper_1006_0663_b200 import inputs
    g = make_solver(teuk, w, options, steps)
    host_in = torch.from_numpy(inputs.initial_state(w)).pin_memory()
    host_out = torch.empty((4, w.precision, w.n_theta, w.n_r), dtype=torch.float64).pin_memory()
    g.set_initial_pinned(host_in)
    g.step(min(steps, 64))
    g.read_pinned(host_out)                     # warm-up of the whole call sequence
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    g.set_initial_pinned(host_in)
    g.step(steps)
    g.read_pinned(host_out)                     # synchronises the stream
    dt = time.perf_counter() - t0
    g.close()
    return dt, host_in.numel() * 8, host_out.numel() * 8


def cpu_baseline(w):
    """the oracle as it stands, on this box's host cores, on a bounded sample of the same workload."""
    import numpy as np
    from oracle import oracle
    from paper_1006_0663_b200 import inputs
    n_win = min(w.n_r, 1024)
    i_lo = max(0, int((inputs.pulse_parameters(w)[0] - w.rstar_min) / w.dr) - n_win // 2)
    cores = oracle.set_threads(0)
    o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win)
    o.set_initial(np.ascontiguousarray(inputs.initial_state(w)[..., i_lo:i_lo + n_win]))
    steps = {1: 400, 2: 8, 4: 4}[w.precision]
    o.step(2)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    # the same sample on ONE host thread (single-core and all-core figures side by side)
    oracle.set_threads(1)
    s1 = max(1, steps // 8)
    t1 = time.perf_counter()
    o.step(s1)
    dt1 = time.perf_counter() - t1
    oracle.set_threads(cores)
    return {"value": n_win * w.n_theta * steps / dt, "unit": "updates/s", "cores": cores, "kind": "oracle",
            "sample": f"radial window of {n_win} of {w.n_r} columns x {w.n_theta} rows, {steps} steps, {w.name}",
            "single_core_value": n_win * w.n_theta * s1 / dt1}


def load_traffic(name):
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(name)
    except Exception:
        return None


def run_sweep(args):
    """BASELINE.json config 5 (a = 0.99, s = -2, m = 2): updates/s and roofline fraction per cell.  fp64: HBM fraction
    (192 B/update vs MEASURED_PEAKS hbm_gbs); dd/qd: FP64-pipe fraction = measured FP64 thread instructions per update
    (ncu, profiles/r01b_step_kernels_ncu.md: 1294 dd, 13320 qd FP64 instructions per update (profiles/r01c_dd_qd_ncu.md), redundant halo work included) x updates/s / measured DFMA-chain peak."""
    import torch
    from paper_1006_0663_b200 import teuk
    torch.cuda.set_device(0)
    peak, _ = measured_peaks()
    pipe = teuk.bench_fp64("dadd")
    inst = FP64_INST_PER_UPDATE
    for L in ((1, 2, 4) if not args.precisions else [int(x) for x in args.precisions.split(",")]):
        for nr in (4096, 16384, 65536):
            for nt in (32, 64, 256):
                w = workload(f"sweep:{nr}x{nt}:{L}")
                steps = {1: 1000, 2: 300, 4: 100}[L] if args.steps == 2000 else args.steps
                ms, launches, geom, finite = time_device(torch, teuk, w, steps, 10, args.option)
                ups = nr * nt * steps / (ms * 1e-3)
                line = {"workload": w.name, "precision_limbs": L, "n_r": nr, "n_theta": nt, "steps": steps,
                        "dt_over_dr": w.dt / w.dr, "updates_per_s": ups, "ms_per_step": ms / steps, "finite": finite,
                        "geometry": geom}
                if L == 1:
                    opt = [o.replace(" ", "") for o in args.option]
                    bpu = 80.0 if "coef_variant=1" in opt else 64.0 if "coef_variant=2" in opt else 96.0 if "time_block=2" in opt else 192.0
                    line["roofline"] = {"bound": "hbm", "frac": ups * bpu / 1e9 / peak, "peak_gbs": peak,
                                        "algorithmic_bytes_per_update": bpu,
                                        "working_set_mib": 24 * nr * nt * 8 // 2 ** 20}
                else:
                    line["roofline"] = {"bound": "fp64 pipe", "frac": ups * inst[L] / pipe, "peak_inst_per_s": pipe,
                                        "fp64_inst_per_update": inst[L]}
                print(json.dumps(line), flush=True)


def run_slabs(args):
    """--shard slabs: the workload's grid cut into world_size r* slabs, one per GPU; each rank steps its window and swaps
    halo strips with its neighbours (NCCL point-to-point) once per 32 iterations.  value = the WHOLE grid's updates / max
    over ranks of the device time (strong scaling); redundant halo columns are not counted as updates."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1006_0663_b200 import inputs, replicas, slabs
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    d = None
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        d = dist
    w = workload(args.workload)
    every = 32
    slab = slabs.plan(w.n_r, world, every)[rank]
    opts = {k: float(v) for k, _, v in (o.partition("=") for o in args.option)}
    u0 = np.ascontiguousarray(inputs.initial_state(w)[..., slab.wlo:slab.whi])
    host_in = torch.from_numpy(u0).pin_memory()
    host_out = torch.empty((4, w.precision, w.n_theta, slab.n_win), dtype=torch.float64).pin_memory()

    def one_run(steps, through_host):
        st = slabs.TeukStepper(w, slab, options=opts, device=f"cuda:{local}")
        run = slabs.SlabRun(slab, st, d, exchange_every=every)
        st.g.set_initial_pinned(host_in)
        run.step(args.warmup)
        torch.cuda.synchronize()
        if d is not None:
            d.barrier()
        n0 = st.g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        if through_host:
            st.g.set_initial_pinned(host_in)
        e0.record(st.g.stream)
        run.step(steps)
        e1.record(st.g.stream)                  # the last exchange ends with write_columns on this stream
        if through_host:
            st.g.read_pinned(host_out)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        res = (e0.elapsed_time(e1), wall, st.g.launch_count() - n0, st.g.step_geometry(), run.exchanges)
        st.g.close()
        return res

    with ClockSampler(local) as cs:
        ms, _, launches, geom, exch = one_run(args.steps, False)
    _, wall, _, _, _ = one_run(args.steps, True)
    points = float(w.n_r * w.n_theta)
    # every rank reports its share of the grid's updates; aggregate() sums them and takes the max time
    mine = float((slab.hi - slab.lo) * w.n_theta) * args.steps
    ms_max, _, value = replicas.aggregate(ms, mine, d, device="cuda")
    _, _, e2e_val = replicas.aggregate(wall * 1e3, mine, d, device="cuda")
    if rank == 0:
        peak, peak_src = measured_peaks()
        L = w.precision
        ach = ALG_BYTES_PER_UPDATE[L] * (slab.n_win * w.n_theta) / (ms / args.steps * 1e-3) / 1e9
        print(json.dumps({
            "metric": "Teukolsky grid-point updates/s", "value": value, "unit": "updates/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": {1: "f64", 2: "f64x2 (double-double)", 4: "f64x4 (quad-double)"}[L],
            "data": "synthetic",
            "config": {"workload": w.name, "n_r": w.n_r, "n_theta": w.n_theta, "precision_limbs": L,
                       "parallelism": f"r*-slabs x{world}, halo {slab.halo}, one exchange per {every} iterations",
                       "rank0_window_columns": slab.n_win, "geometry": geom, "halo_exchanges": exch,
                       "l2": "per-rank working set shrinks with N; no flush (strong scaling of the named workload)"},
            "clocks": cs.summary(),
            "e2e": {"value": e2e_val, "unit": "updates/s", "h2d_bytes_per_step": host_in.numel() * 8 / args.steps,
                    "d2h_bytes_per_step": host_out.numel() * 8 / args.steps},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm" if L == 1 else "fp64 pipe (see profiles/)", "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": None, "peak_source": peak_src,
                         "note": "rank 0's window incl. halo columns"}}), flush=True)
    if d is not None:
        d.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.shard == "slabs":
        return run_slabs(args)
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    d = None
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        d = dist
    from paper_1006_0663_b200 import teuk
    w = workload(args.workload)
    L = w.precision
    points = w.n_r * w.n_theta
    with ClockSampler(local) as cs:
        ms, launches, geom, finite = time_device(torch, teuk, w, args.steps, args.warmup, args.option, d)
    clocks = cs.summary()
    from paper_1006_0663_b200 import replicas
    # max over ranks of the device time, updates summed over ranks; replicas only, no data-path collective
    ms_max, _, value = replicas.aggregate(ms, float(points) * args.steps, d, device="cuda")
    e2e_dt, h2d, d2h = time_e2e(torch, teuk, w, args.steps, args.option)
    _, _, e2e_val = replicas.aggregate(e2e_dt * 1e3, float(points) * args.steps, d, device="cuda")
    if rank != 0:
        if d is not None:
            d.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    opt_set = {o.replace(" ", "") for o in args.option}
    recompute = "coef_variant=1" in opt_set or "coef_variant=2" in opt_set
    # H1b variant (b): state 64 B + two 1/Sigma planes 16 B; (c): state only; NEXT-3: half of the stored-plane traffic
    bytes_per_update = (80.0 if "coef_variant=1" in opt_set else 64.0 if "coef_variant=2" in opt_set
                        else 96.0 if "time_block=2" in opt_set and L == 1 else ALG_BYTES_PER_UPDATE[L])
    alg_bytes = bytes_per_update * points
    achieved = alg_bytes / (ms / args.steps * 1e-3) / 1e9
    line = {
        "metric": "Teukolsky grid-point updates/s", "value": value, "unit": "updates/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None,
        "dtype": {1: "f64", 2: "f64x2 (double-double)", 4: "f64x4 (quad-double)"}[L], "data": "synthetic",
        "config": {"workload": w.name, "M": w.M, "a": w.a, "s": w.s, "m": w.m, "n_r": w.n_r, "n_theta": w.n_theta,
                   "dt_over_dr": w.dt / w.dr, "precision_limbs": L, "parallelism": f"replicas x{world}",
                   "l2": "working set (2 state copies + 16L coefficient planes = %d MiB) exceeds the 126 MB L2; no flush"
                         % (24 * L * points * 8 // 2 ** 20),
                   "geometry": geom, "finite": finite},
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": "updates/s", "h2d_bytes_per_step": h2d / args.steps,
                "d2h_bytes_per_step": d2h / args.steps,
                "note": "teuk_set_initial(host) + teuk_step(K) + teuk_read(host) timed by wall clock; bytes are the whole "
                        "state once per K-step call divided by K"},
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": load_traffic(f"{w.name}"), "peak_source": peak_src, "kernel": "step_kernel_f64_rc" if recompute else ("step2_kernel_f64_tma" if "time_block=2" in opt_set and L == 1 else "step_kernel_f64_tma" if L == 1 else f"step_kernel<{L}>"),
                     "algorithmic_bytes_per_update": bytes_per_update},
    }
    if not args.no_extra and world == 1:
        per = {}
        fp = {k: teuk.bench_fp64(k) for k in ("dfma", "dadd", "dmul")}
        for name, k_steps in (("cfg3", max(50, args.steps // 10)), ("cfg4", max(50, args.steps // 10))):
            wx = workload(name)
            msx, lx, gx, fx = time_device(torch, teuk, wx, k_steps, 20, args.option)
            upsx = wx.n_r * wx.n_theta * k_steps / (msx * 1e-3)
            per[name] = {"precision_limbs": wx.precision, "n_r": wx.n_r, "n_theta": wx.n_theta, "steps": k_steps,
                         "updates_per_s": upsx, "ms_per_step": msx / k_steps, "geometry": gx, "finite": fx,
                         # FP64 instructions per update from ncu (profiles/r01e_step_kernels_ncu.md) x rate / measured DADD issue peak
                         "roofline": {"bound": "fp64 pipe", "fp64_inst_per_update": FP64_INST_PER_UPDATE[wx.precision],
                                      "peak_inst_per_s": fp["dadd"], "frac": upsx * FP64_INST_PER_UPDATE[wx.precision] / fp["dadd"]}}
        # NEXT-1: the same three workloads with the 10th-order theta operator (column kernel)
        t10 = {}
        for name, k_steps in (("cfg2", max(50, args.steps // 10)), ("cfg3", max(50, args.steps // 10)), ("cfg4", max(50, args.steps // 10))):
            wx = workload(name)
            wx = wx.scaled(dt_override=0.5 * wx.dt)
            msx, lx, gx, fx = time_device(torch, teuk, wx, k_steps, 20, list(args.option) + ["theta_order=10"])
            t10[name] = {"precision_limbs": wx.precision, "steps": k_steps, "updates_per_s": wx.n_r * wx.n_theta * k_steps / (msx * 1e-3),
                         "ms_per_step": msx / k_steps, "geometry": gx, "finite": fx}
        line["theta_order_10"] = t10
        # H1b variant (b): semi-recompute coefficient supply for the primary workload (80 B/update)
        if L == 1:
            msr, lr, gr, fr = time_device(torch, teuk, w, args.steps, args.warmup, list(args.option) + ["coef_variant=1"])
            ach = 80.0 * points / (msr / args.steps * 1e-3) / 1e9
            line["semi_recompute"] = {"updates_per_s": points * args.steps / (msr * 1e-3), "ms_per_step": msr / args.steps,
                                      "algorithmic_bytes_per_update": 80.0, "hbm_frac": ach / peak, "geometry": gr, "finite": fr}
            # H1b variant (c): full recompute (1/Sigma by rsqrt per point; state-only traffic, 64 B/update)
            msf, lf, gf, ff = time_device(torch, teuk, w, args.steps, args.warmup, list(args.option) + ["coef_variant=2"])
            achf = 64.0 * points / (msf / args.steps * 1e-3) / 1e9
            line["full_recompute"] = {"updates_per_s": points * args.steps / (msf * 1e-3), "ms_per_step": msf / args.steps,
                                      "algorithmic_bytes_per_update": 64.0, "hbm_frac": achf / peak, "geometry": gf, "finite": ff}
            # NEXT-3: two iterations per launch (u^{n+1} and the coefficient tiles stay on the SM): 96 B/update
            mst, lt, gt, ft = time_device(torch, teuk, w, args.steps, args.warmup, list(args.option) + ["time_block=2"])
            acht = 96.0 * points / (mst / args.steps * 1e-3) / 1e9
            line["time_blocked_2"] = {"updates_per_s": points * args.steps / (mst * 1e-3), "ms_per_step": mst / args.steps,
                                      "algorithmic_bytes_per_update": 96.0, "hbm_frac": acht / peak, "gpu_launches": lt,
                                      "geometry": gt, "finite": ft}
        line["per_precision"] = per
        line["fp64_pipe_peak_inst_per_s"] = fp
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line), flush=True)
    if d is not None:
        d.destroy_process_group()


if __name__ == "__main__":
    main()
