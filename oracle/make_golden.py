"""ORACLE (test infrastructure, not product code) -- writes the cached full-length oracle results that the
`-m gpu` parity tests compare with (tests/golden/cfg{2,3,4}_full.npz; SURVEY.md 8(d) "Full-length oracle runs are for
parity only and are cached on disk"; BASELINE.json `north_star`: "GPU results must match the oracle ... after the run").

It imports only `oracle/` and the seeded input recipe (`paper_1006_0663_b200/inputs.py`, no method arithmetic);
nothing here touches the CUDA path.  fp64 runs use the plain double stepper, dd/qd runs the fast arithmetic tier
(oracle/mpf.hpp), which is pinned operation by operation against the exact-then-round tier.

    python -m oracle.make_golden --cfg 3 --threads 8            # hours for cfg 3 / cfg 4: run in the background

The run advances the FULL grid (no window) in chunks, keeps a resume file after every chunk (--resume-dir, default
/tmp/teuk_golden) and rewrites the output after every stored checkpoint, so an interrupted run leaves a usable
prefix.  Stored per config:
    meta          json: parameters, dt, precision, tier, column strides, sha256 of the oracle sources, `git rev-parse HEAD:oracle`
    observer      [steps_done][4][L]   the observer series in full, all limbs
    checkpoints   [k]                  step counts at which the state was sampled (the last one = steps_done)
    state_<n>     [4][L][N_theta][n_cols]  every `stride`-th r* column of the state after n steps, all limbs
                  (stride 8 at the last checkpoint of a completed run, 64 at the intermediate ones: 10 %, 20 %, 25 %, ...
                  of the run; a run that was resumed under an older version of this script may lack some of them)
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import time

import numpy as np

from paper_1006_0663_b200 import inputs

from . import oracle

_HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["teuk_oracle.cpp", "mpx.hpp", "mpf.hpp", "mp_ref.py"]
FINAL_STRIDE, MID_STRIDE = 8, 64
# step counts at which the state is sampled (fractions of the run), the last one being the full length
CHECKPOINT_FRACTIONS = (0.1, 0.2, 0.25, 0.3, 0.4, 0.5, 0.6, 0.7, 0.75, 0.8, 0.9, 1.0)


def source_hash() -> str:
    h = hashlib.sha256()
    for name in SOURCES:
        with open(os.path.join(_HERE, name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def git_tree() -> str:
    try:
        return subprocess.check_output(["git", "rev-parse", "HEAD:oracle"], cwd=_HERE, text=True,
                                       stderr=subprocess.DEVNULL).strip()
    except Exception:
        return "unknown"


def checkpoints(steps: int) -> list:
    return sorted({max(1, int(round(f * steps))) for f in CHECKPOINT_FRACTIONS})


def golden_path(k: int, out_dir: str) -> str:
    return os.path.join(out_dir, f"cfg{k}_full.npz")


def write(path, meta, series, samples):
    arrays = {"meta": np.array(json.dumps(meta)), "observer": series,
              "checkpoints": np.array(sorted(samples), dtype=np.int64)}
    for n, arr in samples.items():
        arrays[f"state_{n}"] = arr
    tmp = path + ".tmp.npz"
    np.savez(tmp, **arrays)
    os.replace(tmp, path)


def run(k: int, out_dir: str, resume_dir: str, threads: int, chunk: int, max_steps: int | None):
    w = inputs.config(k)
    steps = w.steps if max_steps is None else min(w.steps, max_steps)
    tier = "exact" if w.precision == 1 else "fast"
    used = oracle.set_threads(threads)
    ro, to = w.observer
    meta = {"config": k, "M": w.M, "a": w.a, "s": w.s, "m": w.m, "n_r": w.n_r, "n_theta": w.n_theta,
            "rstar_min": w.rstar_min, "rstar_max": w.rstar_max, "dt": w.dt, "dt_hex": float(w.dt).hex(),
            "steps_full": w.steps, "precision": w.precision, "tier": tier, "seed": w.seed,
            "observer": [ro, to], "final_stride": FINAL_STRIDE, "mid_stride": MID_STRIDE,
            "oracle_sources": SOURCES, "oracle_sha256": source_hash(), "oracle_git_tree": git_tree(), "threads": used}
    os.makedirs(resume_dir, exist_ok=True)
    os.makedirs(out_dir, exist_ok=True)
    rfile = os.path.join(resume_dir, f"cfg{k}_resume.npz")
    t0 = time.time()
    o = oracle.Oracle.from_workload(w, tier=tier)
    print(f"cfg{k}: tables built in {time.time() - t0:.0f} s, {used} threads, tier {tier}", flush=True)
    done, series, samples = 0, np.zeros((0, 4, w.precision)), {}
    if os.path.exists(rfile):
        with np.load(rfile) as z:
            if str(z["sha"]) == meta["oracle_sha256"] and float(z["dt"]) == w.dt:
                done, series = int(z["done"]), z["series"]
                samples = {int(n): z[f"state_{n}"] for n in z["checkpoints"]}
                o.set_initial(z["state"])
                print(f"cfg{k}: resumed at step {done}", flush=True)
    if done == 0:
        o.set_initial(inputs.initial_state(w))
    marks = [c for c in checkpoints(w.steps) if c <= steps]
    if steps not in marks:
        marks.append(steps)
    t0, start = time.time(), done
    while done < steps:
        nxt = min([c for c in marks if c > done] + [done + chunk])
        n = nxt - done
        o.set_observer(ro, to, n)            # restarts the series buffer; samples are appended below
        o.step(n)
        series = np.concatenate([series, o.observe(n)])
        done = nxt
        state = o.read()
        if done in marks:
            stride = FINAL_STRIDE if done == w.steps else MID_STRIDE
            samples[done] = np.ascontiguousarray(state[:, :, :, ::stride])
            meta["steps_done"] = done
            write(golden_path(k, out_dir), meta, series, samples)
        np.savez(rfile + ".tmp.npz", sha=meta["oracle_sha256"], dt=w.dt, done=done, series=series, state=state,
                 checkpoints=np.array(sorted(samples), dtype=np.int64),
                 **{f"state_{n}": a for n, a in samples.items()})
        os.replace(rfile + ".tmp.npz", rfile)
        el = time.time() - t0
        rate = (done - start) * w.n_r * w.n_theta / max(el, 1e-9)
        eta = (steps - done) * w.n_r * w.n_theta / max(rate, 1.0)
        print(f"cfg{k}: step {done}/{steps}  {rate:.3e} updates/s  elapsed {el / 60:.1f} min  eta {eta / 60:.1f} min",
              flush=True)
    print(f"cfg{k}: wrote {golden_path(k, out_dir)}", flush=True)


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--cfg", type=int, nargs="+", default=[2, 3, 4])
    ap.add_argument("--out", default=os.path.join(os.path.dirname(_HERE), "tests", "golden"))
    ap.add_argument("--resume-dir", default="/tmp/teuk_golden")
    ap.add_argument("--threads", type=int, default=0, help="OpenMP threads (0 = all)")
    ap.add_argument("--chunk", type=int, default=500, help="steps between resume files")
    ap.add_argument("--max-steps", type=int, default=None, help="stop early (stores the prefix reached)")
    a = ap.parse_args()
    for k in a.cfg:
        run(k, a.out, a.resume_dir, a.threads, a.chunk, a.max_steps)


if __name__ == "__main__":
    main()
