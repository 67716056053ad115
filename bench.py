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

ALG_BYTES_PER_UPDATE = {1: 192.0, 2: 384.0, 4: 768.0}     # DESIGN.md §6, stored planes: 4L read + 4L write + 16L coefficients, x 8 B
SEMI_RECOMPUTE_BYTES = 80.0                               # fp64 semi-recompute supply: 64 B of state + two 1/Sigma values
FALLBACK_HBM_GBS = 6650.0
REPS = 5                                                  # timed repetitions of the K-step region; median and min are reported
DTYPE = {1: "f64", 2: "f64x2 (double-double)", 4: "f64x4 (quad-double)"}


def fp64_inst_per_update():
    """FP64 (DADD + DMUL + DFMA) thread instructions per update of the dd / qd step kernels: `measured` = ncu count of the
    kernel as built (redundant halo half steps included), `method` = the count of the update itself (no halo work).
    Written next to the ncu summary it comes from (profiles/fp64_inst.json names the capture and the csrc/ revision)."""
    with open(os.path.join(ROOT, "profiles", "fp64_inst.json")) as f:
        d = json.load(f)
    return {(2, 2): d["dd"], (4, 2): d["qd"], (2, 10): d["dd_theta10"], (4, 10): d["qd_theta10"]}


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
    o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win, tier="exact" if w.precision == 1 else "fast")
    u0 = inputs.initial_state(w)[..., i_lo:i_lo + n_win]
    o.set_initial(np.ascontiguousarray(u0))
    o.step(args.warmup if w.precision == 1 else min(args.warmup, 2))
    steps = args.steps if w.precision == 1 else max(1, min(args.steps, 40))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    val = n_win * w.n_theta * steps / dt
    sample = f"radial window of {n_win} of {w.n_r} columns x {w.n_theta} rows, {steps} steps"
    line = {"impl": "reference", "metric": "Teukolsky grid-point updates/s", "value": val, "unit": "updates/s",
            "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": DTYPE[w.precision],
            "data": "synthetic", "config": {"workload": w.name, "n_r": w.n_r, "n_theta": w.n_theta,
                                            "dt_over_dr": w.dt / w.dr, "sample": sample},
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


_flush_buf = None


def flush_l2(torch, device):
    """write a buffer larger than the 126 MB L2 (between timed repetitions)"""
    global _flush_buf
    if _flush_buf is None or _flush_buf.device != torch.device(device):
        _flush_buf = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=device)
    _flush_buf.fill_(1)


def time_device(torch, teuk, w, steps, warmup, options, dist=None, reps=REPS):
    """inputs resident in HBM; CUDA events on the stream the kernels are launched on.  W untimed warm-up iterations and one
    untimed K-iteration call (which instantiates the CUDA graph of that call), then REPS timed repetitions of exactly K
    iterations each, L2 flushed between repetitions.  Returns the median repetition (ms) and the rest beside it."""
    from paper_1006_0663_b200 import inputs
    g = make_solver(teuk, w, options, warmup + steps * (reps + 1))
    u0 = torch.from_numpy(inputs.initial_state(w)).to(g.device)
    g.set_initial(u0)
    g.step(warmup)
    g.step(steps)
    torch.cuda.synchronize()
    times, launches = [], 0
    for _ in range(reps):
        flush_l2(torch, g.device)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        n0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(g.stream)
        g.step(steps)
        e1.record(g.stream)
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
        if dist is not None:
            dist.barrier()
        launches = g.launch_count() - n0
    geom = g.step_geometry()
    g.observe(4, allow_nonfinite=True)
    finite = bool(torch.isfinite(g.read_device()).all().item()) and g.last_observe_status == 0
    g.close()
    ts = sorted(times)
    return {"ms": ts[len(ts) // 2], "ms_min": ts[0], "ms_all": times, "launches": launches, "geometry": geom, "finite": finite}


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
    """the oracle as it stands, on this box's host cores, on a bounded sample of the same workload (fp64: the plain
    double stepper; dd/qd: its fast arithmetic tier, the one the full-length golden runs use)."""
    import numpy as np
    from oracle import oracle
    from paper_1006_0663_b200 import inputs
    n_win = min(w.n_r, 1024)
    i_lo = max(0, int((inputs.pulse_parameters(w)[0] - w.rstar_min) / w.dr) - n_win // 2)
    cores = oracle.set_threads(0)
    tier = "exact" if w.precision == 1 else "fast"
    o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win, tier=tier)
    o.set_initial(np.ascontiguousarray(inputs.initial_state(w)[..., i_lo:i_lo + n_win]))
    o.step(2)
    # size the sample for a few seconds of CPU work from a short probe
    t0 = time.perf_counter()
    o.step(2)
    probe = (time.perf_counter() - t0) / 2
    steps = int(max(4, min(2000, 5.0 / max(probe, 1e-6))))
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
    return {"value": n_win * w.n_theta * steps / dt, "unit": "updates/s", "cores": cores, "kind": "oracle", "tier": tier,
            "sample": f"radial window of {n_win} of {w.n_r} columns x {w.n_theta} rows, {steps} steps, {w.name}",
            "single_core_value": n_win * w.n_theta * s1 / dt1}


def load_traffic(name):
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(p)).get(name)
    except Exception:
        return None


def supply_of(options, L):
    """(label, algorithmic bytes per update) of the coefficient supply the option list selects"""
    opt = {o.replace(" ", "") for o in options}
    if L == 1 and ("coef_variant=1" in opt or ("theta_order=10" in opt and "use_tma=0" not in opt)):
        return "semi_recompute", SEMI_RECOMPUTE_BYTES      # the fp64 10th-order column kernel always uses this supply
    if L == 1 and "coef_variant=2" in opt:
        return "full_recompute", 64.0
    if L == 1 and "time_block=2" in opt:
        return "stored_planes_time_block_2", 96.0
    return "stored_planes", ALG_BYTES_PER_UPDATE[L]


def hbm_roofline(ups, points, bytes_per_update, peak, peak_src, kernel, traffic=None):
    achieved = ups * bytes_per_update / 1e9
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
            "peak_source": peak_src, "kernel": kernel, "algorithmic_bytes_per_update": bytes_per_update,
            "algorithmic_bytes_per_launch": bytes_per_update * points}


def pipe_roofline(ups, L, pipe_peak, theta_order=2):
    inst = fp64_inst_per_update()[(L, theta_order)]
    return {"bound": "alu", "pipe": "fp64", "achieved": ups * inst["measured"], "peak": pipe_peak, "unit": "FP64 inst/s",
            "frac": ups * inst["measured"] / pipe_peak, "frac_method_only": ups * inst["method"] / pipe_peak,
            "fp64_inst_per_update_measured": inst["measured"], "fp64_inst_per_update_method": inst["method"],
            "inst_source": inst.get("source"), "peak_source": "teuk_bench_fp64 DADD chains, this run", "traffic": None}


def kernel_name(L, options):
    opt = {o.replace(" ", "") for o in options}
    if "theta_order=10" in opt:
        if L == 1:
            return "step_kernel_col<1>" if "use_tma=0" in opt else ("step_kernel_f64_col_tma" if "col_run=0" in opt else "step_kernel_f64_col_run")
        return "step_kernel_col_pair<4>" if (L == 4 and "variant=4" not in opt) else f"step_kernel_col<{L}>"
    if L == 1:
        if "coef_variant=1" in opt:
            return "step_kernel_f64_rc" if "march=0" in opt else "step_kernel_f64_march"
        if "coef_variant=2" in opt:
            return "step_kernel_f64_rc<full>"
        return "step2_kernel_f64_tma" if "time_block=2" in opt else "step_kernel_f64_tma"
    if L == 4 and "variant=4" not in opt:
        return "step_kernel_pair<4>"
    return f"step_kernel<{L}>"


def run_sweep(args):
    """BASELINE.json config 5 (a = 0.99, s = -2, m = 2): updates/s and roofline fraction per cell.  fp64: HBM fraction of
    the selected coefficient supply; dd/qd: FP64-pipe fraction = FP64 thread instructions per update (profiles/fp64_inst.json)
    x updates/s / DADD issue rate measured in this run."""
    import torch
    from paper_1006_0663_b200 import teuk
    torch.cuda.set_device(0)
    peak, peak_src = measured_peaks()
    pipe = teuk.bench_fp64("dadd")
    for L in ((1, 2, 4) if not args.precisions else [int(x) for x in args.precisions.split(",")]):
        for nr in (4096, 16384, 65536):
            for nt in (32, 64, 256):
                w = workload(f"sweep:{nr}x{nt}:{L}")
                steps = {1: 400, 2: 120, 4: 40}[L] if args.steps == 2000 else args.steps
                opts = list(args.option)
                if L == 1 and not any(o.replace(" ", "").startswith("coef_variant") for o in opts):
                    opts.append("coef_variant=1")      # explicit, so that the line is labelled with the supply that ran
                r = time_device(torch, teuk, w, steps, 10, opts, reps=3)
                ups = nr * nt * steps / (r["ms"] * 1e-3)
                label, bpu = supply_of(opts, L)
                line = {"workload": w.name, "precision_limbs": L, "n_r": nr, "n_theta": nt, "steps": steps,
                        "dt_over_dr": w.dt / w.dr, "updates_per_s": ups, "ms_per_step": r["ms"] / steps,
                        "ms_per_step_min": r["ms_min"] / steps, "finite": r["finite"], "geometry": r["geometry"],
                        "supply": label}
                if L == 1:
                    line["roofline"] = hbm_roofline(ups, nr * nt, bpu, peak, peak_src, kernel_name(L, opts))
                    line["working_set_mib"] = int((bpu + 64) * nr * nt) // 2 ** 20
                else:
                    line["roofline"] = pipe_roofline(ups, L, pipe, 10 if "theta_order=10" in args.option else 2)
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
        ach = supply_of(args.option, L)[1] * (slab.n_win * w.n_theta) / (ms / args.steps * 1e-3) / 1e9
        print(json.dumps({
            "metric": "Teukolsky grid-point updates/s", "value": value, "unit": "updates/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": DTYPE[L],
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


def measure(torch, teuk, name, steps, warmup, options, peak, peak_src, pipe, dist=None, with_cpu=True, with_e2e=True):
    """one workload: device-timed rate (median of REPS), roofline of its step kernel, e2e through host buffers, oracle beside it"""
    w = workload(name) if isinstance(name, str) else name
    L, points = w.precision, w.n_r * w.n_theta
    r = time_device(torch, teuk, w, steps, warmup, options, dist)
    ups = points * steps / (r["ms"] * 1e-3)
    label, bpu = supply_of(options, L)
    out = {"workload": w.name, "precision_limbs": L, "dtype": DTYPE[L], "n_r": w.n_r, "n_theta": w.n_theta,
           "dt_over_dr": w.dt / w.dr, "baseline_dt_over_dr": 0.5, "steps": steps, "updates_per_s": ups,
           "ms_per_step": r["ms"] / steps, "ms_per_step_min": r["ms_min"] / steps,
           "ms_per_step_all": [t / steps for t in r["ms_all"]], "gpu_launches": r["launches"], "geometry": r["geometry"],
           "finite": r["finite"], "coefficient_supply": label}
    kern = kernel_name(L, options)
    if L == 1:
        out["roofline"] = hbm_roofline(ups, points, bpu, peak, peak_src, kern, load_traffic(f"{w.name}:{kern}"))
        out["working_set_mib"] = int((bpu + 64) * points) // 2 ** 20
    else:
        out["roofline"] = pipe_roofline(ups, L, pipe, 10 if "theta_order=10" in options else 2)
        out["roofline"]["kernel"] = kern
        out["roofline"]["traffic"] = load_traffic(f"{w.name}:{kern}")
        out["hbm_frac_at_this_rate"] = ups * ALG_BYTES_PER_UPDATE[L] / 1e9 / peak
    if with_e2e:
        dt, h2d, d2h = time_e2e(torch, teuk, w, steps, options)
        out["e2e"] = {"value": points * steps / dt, "unit": "updates/s", "h2d_bytes_per_step": h2d / steps,
                      "d2h_bytes_per_step": d2h / steps}
    if with_cpu:
        out["cpu_baseline"] = cpu_baseline(w)
    return out, r


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
    from paper_1006_0663_b200 import replicas, teuk
    w = workload(args.workload)
    L = w.precision
    points = w.n_r * w.n_theta
    # headline path for fp64: the semi-recompute coefficient supply (H1b variant (b), 80 B/update) unless the caller chose
    # a supply; dd/qd: stored planes (they are FP64-pipe bound)
    opts = list(args.option)
    chose = any(o.replace(" ", "").split("=")[0] in ("coef_variant", "time_block", "use_tma", "theta_order") for o in opts)
    if L == 1 and not chose:
        opts.append("coef_variant=1")
    other = [o for o in opts if not o.replace(" ", "").startswith("coef_variant")]
    peak, peak_src = measured_peaks()
    pipe = teuk.bench_fp64("dadd")
    extra = not args.no_extra and world == 1
    with ClockSampler(local) as cs:
        head, r = measure(torch, teuk, w, args.steps, args.warmup, opts, peak, peak_src, pipe, d,
                          with_cpu=extra and rank == 0, with_e2e=False)
    clocks = cs.summary()
    # max over ranks of the device time, updates summed over ranks; replicas only, no data-path collective
    ms_max, _, value = replicas.aggregate(r["ms"], float(points) * args.steps, d, device="cuda")
    e2e_dt, h2d, d2h = time_e2e(torch, teuk, w, args.steps, opts)
    _, _, e2e_val = replicas.aggregate(e2e_dt * 1e3, float(points) * args.steps, d, device="cuda")
    if rank != 0:
        if d is not None:
            d.destroy_process_group()
        return
    label, bpu = supply_of(opts, L)
    ws_mib = int(((bpu + 64) if L == 1 else 24 * 8 * L) * points) // 2 ** 20
    line = {
        "metric": "Teukolsky grid-point updates/s", "value": value, "unit": "updates/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE[L], "data": "synthetic",
        "config": {"workload": w.name, "M": w.M, "a": w.a, "s": w.s, "m": w.m, "n_r": w.n_r, "n_theta": w.n_theta,
                   "dt_over_dr": w.dt / w.dr, "baseline_dt_over_dr": 0.5,
                   "dt_note": "BASELINE.json says dt = 0.5 dr*; configs 2/3/5 are unstable there (DESIGN.md reading A15b, "
                              "tests/test_oracle_stability.py) and run at inputs.stable_dt; work per update is unchanged",
                   "precision_limbs": L, "parallelism": f"replicas x{world}", "coefficient_supply": label, "options": opts,
                   "timing": f"median of {REPS} repetitions of {args.steps} iterations (min and all repetitions under "
                             "ms_per_step_min / ms_per_step_all); one CUDA-graph launch per teuk_step call",
                   "l2": f"L2 flushed (256 MiB write) between timed repetitions; inside a repetition the time loop re-reads "
                         f"its own working set of {ws_mib} MiB (L2 is 126 MB): the HBM-bound claim is made on `large_cell`",
                   "geometry": head["geometry"], "finite": head["finite"]},
        "ms_per_step_min": head["ms_per_step_min"], "ms_per_step_all": head["ms_per_step_all"],
        "clocks": clocks,
        "e2e": {"value": e2e_val, "unit": "updates/s", "h2d_bytes_per_step": h2d / args.steps,
                "d2h_bytes_per_step": d2h / args.steps,
                "note": "teuk_set_initial(host) + teuk_step(K) + teuk_read(host) timed by wall clock; bytes are the whole "
                        "state once per K-step call divided by K"},
        "gpu_launches": r["launches"],
        "roofline": head["roofline"],
    }
    if extra:
        line["cpu_baseline"] = head["cpu_baseline"]
        k10 = max(50, args.steps // 10)
        if L == 1 and not chose:
            # the other coefficient supply of the primary workload (H1b): stored planes, 192 B/update
            line["stored_planes"], _ = measure(torch, teuk, w, args.steps, args.warmup, other + ["coef_variant=0"],
                                               peak, peak_src, pipe, with_cpu=False, with_e2e=False)
            # above L2: sweep cell 65536 x 64 (working set 576 MiB semi-recompute / 1 GiB stored planes), both supplies
            big = {}
            for tag, o2 in (("semi_recompute", ["coef_variant=1"]), ("stored_planes", ["coef_variant=0"])):
                big[tag], _ = measure(torch, teuk, "sweep:65536x64", max(20, args.steps // 4), 10, other + o2,
                                      peak, peak_src, pipe, with_cpu=False, with_e2e=False)
            line["large_cell"] = big
        # dd and qd (BASELINE.json configs[2], configs[3]): rate, FP64-pipe roofline, e2e and the oracle beside each
        per = {}
        for name in ("cfg3", "cfg4"):
            per[name], _ = measure(torch, teuk, name, k10, 20, other, peak, peak_src, pipe)
        line["per_precision"] = per
        # NEXT-1: the same three workloads with the 10th-order theta operator (column kernels)
        t10 = {}
        for name in ("cfg2", "cfg3", "cfg4"):
            wx = workload(name)
            wx = wx.scaled(dt_override=0.5 * wx.dt)
            t10[name], _ = measure(torch, teuk, wx, k10, 20, other + ["theta_order=10"], peak, peak_src, pipe,
                                   with_cpu=False, with_e2e=False)
        line["theta_order_10"] = t10
        line["fp64_pipe_peak_inst_per_s"] = {k: teuk.bench_fp64(k) for k in ("dfma", "dadd", "dmul")}
    print(json.dumps(line), flush=True)
    if d is not None:
        d.destroy_process_group()


if __name__ == "__main__":
    main()
