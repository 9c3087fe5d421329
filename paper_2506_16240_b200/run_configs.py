"""Run BASELINE.json's five configurations at full length on one GPU.

    python -m paper_2506_16240_b200.run_configs [--configs 1 2 3 4 5] [--scale 1.0]

One JSON line per (config, temperature / refresh interval): wall time of the
micsa_anneal call (refreshes, sweeps and measurements, rows read back),
spin-flip attempts per ns, random 32-bit words defined and generated per spin
update, and the physics the config asks for -- energy per spin, daemon energy
per spin, |q| -- at the end of the run (sample average and scatter); for the
annealing config 5 the minimum energy per spin per sample.  `--scale` shortens
every run (0.01 = 1 % of the sweeps) for a quick look.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

from micsa_workloads import CONFIGS, schedule_for
from . import MicSA


def _measure_every(n_sweeps_total, interval):
    """About 100 rows per run, always at the end of a refresh interval."""
    every = max(interval, (n_sweeps_total // 100) // interval * interval)
    return every


def run(ci, scale):
    cfg = CONFIGS[ci]
    N = cfg.N
    cases = []
    if cfg.ramp_steps:
        cases.append(("ramp", None, None))
    else:
        for T in cfg.temperatures:
            for R in cfg.refresh_intervals:
                cases.append((f"T={T}_R={R}", T, R))
    for label, T, R in cases:
        n_sweeps = max(1, int(cfg.n_sweeps * scale))
        if cfg.ramp_steps:
            sched = schedule_for(cfg)
            sched = sched[: max(1, int(len(sched) * scale))] if scale < 1 else sched
        else:
            n_sweeps = max(R, n_sweeps // R * R)
            steps = n_sweeps // R
            me = _measure_every(n_sweeps, R)
            # measure at the end of every k-th refresh interval: measure_every counts sweeps inside a step
            k = max(1, me // R)
            sched = [(float(T), R, R if (i + 1) % k == 0 or i == steps - 1 else 0) for i in range(steps)]
        with MicSA(cfg.L, cfg.n_samples, cfg.n_replicas, cfg.seed) as g:
            g.synchronize()
            t0 = time.perf_counter()
            out = g.anneal(sched)
            dt = time.perf_counter() - t0
            c = g.counters()
        total_sweeps = sum(n for _, n, _ in sched)
        e = out["E"][-1] / N
        ed = out["Edem"][-1] / N
        line = {
            "config": ci, "workload": cfg.name, "case": label, "sweeps": total_sweeps, "refreshes": len(sched),
            "rows": int(out["E"].shape[0]), "wall_s": round(dt, 4),
            "attempts_per_ns": round(c["attempts"] / dt / 1e9, 1),
            "rns_defined_per_attempt": round(c["rns_drawn"] / c["attempts"], 5),
            "philox_words_generated_per_attempt": round(4.0 * c["philox_calls"] / c["attempts"], 5),
            "e_final_mean": round(float(e.mean()), 6), "e_final_scatter": round(float(e.std(ddof=1)) if e.size > 1 else 0.0, 6),
            "e_daemon_final_mean": round(float(ed.mean()), 6),
        }
        if out["Q"].size:
            q = out["Q"][-1] / N
            line["abs_q_final_mean"] = round(float(np.abs(q).mean()), 6)
        if cfg.ramp_steps:
            me_ = out["min_energy"]
            line["min_energy_mean"] = round(float(me_.mean()), 6)
            line["min_energy_best"] = round(float(me_.min()), 6)
            line["T_final"] = sched[-1][0]
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="*", default=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=float, default=1.0)
    args = ap.parse_args()
    for ci in args.configs:
        run(ci, args.scale)


if __name__ == "__main__":
    main()
