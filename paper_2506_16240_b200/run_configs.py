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
from . import GaussMicSA, MicSA, xi as xi_lengths


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
        # a stream above the default priority: the library's side stream (the next refresh) then only fills what
        # the sweeps leave idle (include/micsa.h, micsa_prefetch_refresh)
        import torch
        stream = torch.cuda.Stream(priority=-1)
        with MicSA(cfg.L, cfg.n_samples, cfg.n_replicas, cfg.seed, stream=stream) as warm:   # load the kernels once (lazy module loading)
            warm.anneal(sched[:2], trace=False)
        with MicSA(cfg.L, cfg.n_samples, cfg.n_replicas, cfg.seed, stream=stream) as g:
            g.synchronize()
            t0 = time.perf_counter()
            out = g.anneal(sched)
            dt = time.perf_counter() - t0
            c = g.counters()
            c4 = None
            if cfg.n_replicas >= 2:                      # Eq. (16)-(18) at the end of the run
                S = g.measure_c4().astype(np.float64)
                pps = cfg.n_replicas * (cfg.n_replicas - 1) // 2
                per_sample = S.reshape(cfg.n_samples, pps, 3, -1).sum(axis=(1, 2)) / (3.0 * pps * N)
                c4 = per_sample.mean(axis=0)
                c4_err = per_sample.std(axis=0, ddof=1) / np.sqrt(cfg.n_samples) if cfg.n_samples > 1 else np.zeros_like(c4)
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
        if c4 is not None:
            try:                                         # cut-off: three times the sample error (R22)
                _, _, _, x12, ratio = xi_lengths(c4, float(3.0 * c4_err.max()))
                line["xi12"] = round(x12, 4); line["xi23_over_xi12"] = round(ratio, 4)
            except Exception:
                line["xi12"] = None
        if cfg.ramp_steps:
            me_ = out["min_energy"]
            line["min_energy_mean"] = round(float(me_.mean()), 6)
            line["min_energy_best"] = round(float(me_.min()), 6)
            line["T_final"] = sched[-1][0]
        print(json.dumps(line), flush=True)


def run_gauss(L, n_samples, n_replicas, T, n_emcs, label):
    """Continuous walkers with Gaussian couplings (Appendix C step 1): per EMCS one refresh from Eq. (9) and
    10 x (sweep + forward-X wandering); wall time of the whole loop, energy and |q| at the end."""
    from micsa_workloads import gaussian_couplings
    N = L ** 3
    with GaussMicSA(L, n_samples, n_replicas, 6) as g:
        g.set_couplings(gaussian_couplings((n_samples, 3, N), 7))
        g.set_walkers(1, 0)
        g.refresh(T, 0); g.sweep(10); g.synchronize()
        t0 = time.perf_counter()
        for k in range(1, n_emcs + 1):
            g.refresh(T, k)
            g.sweep(10)
        E, Ed, Q = g.measure()
        dt = time.perf_counter() - t0
        c = g.counters()
    attempts = 10 * n_emcs * N * n_samples * n_replicas
    line = {"config": "appendix_C_move", "workload": f"gauss_L{L}_{n_samples}x{n_replicas}", "case": label, "T": T,
            "sweeps": 10 * n_emcs, "refreshes": n_emcs, "wall_s": round(dt, 4),
            "attempts_per_ns": round(attempts / dt / 1e9, 2),
            "rns_defined_per_attempt": round(c["rns_drawn"] / c["attempts"], 5),
            "e_final_mean": round(float((E / N).mean()), 6), "e_daemon_final_mean": round(float((Ed / N).mean()), 6)}
    if Q.size:
        line["abs_q_final_mean"] = round(float(np.abs(Q / N).mean()), 6)
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="*", default=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--gauss", action="store_true", help="also the continuous-daemon workload (Appendix C move)")
    args = ap.parse_args()
    for ci in args.configs:
        run(ci, args.scale)
    if args.gauss:
        run_gauss(10, 40, 2, 0.2, max(1, int(1000 * args.scale)), "L=10, 40 x 2 systems (the paper's size), T = 0.2")
        run_gauss(64, 32, 2, 1.0, max(1, int(100 * args.scale)), "L=64, 32 x 2 systems, T = 1.0")


if __name__ == "__main__":
    main()
