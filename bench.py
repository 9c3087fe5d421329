#!/usr/bin/env python
"""bench.py -- MicSA hot-path throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl micsa|reference]

One STEP = one pass of the whole hot path over BASELINE
config 4 (L=160, 16 samples x 2 replicas, T=0.9): daemon refresh at T, then
10 checkerboard sweeps, then the E / E_daemon / q reductions.  Prints ONE JSON
line (rank 0).

`value` (attempts per ns, state resident in HBM / L2) is the LOWER of two
device-timed figures, both with a closed timed window:
  * back_to_back: the K steps through ONE micsa_anneal call, one CUDA-event
    pair on the library's stream around all of them (rows read back inside);
  * l2_flushed: K separately timed steps with a 256 MiB write between them
    (outside the events); the window of step k = generation of refresh k+1 on
    the side stream (queued first, consumed last) + 20 half-sweeps + the
    measurement, so no refresh work runs between two windows.
`e2e` = upload of spins and couplings from pinned host int8 arrays once, then
the K steps through micsa_anneal with the rows copied back, wall clock.
`roofline` = the plain half-sweep launches inside the flushed steps;
`hbm_resident` = the same kernels on 160^3 x 128 systems (the shape of the
paper's Table 3; 295 MB of state, larger than L2).
N > 1: one process per GPU (torchrun), samples sharded by rank with global
sample offsets, no data-path collective (weak scaling).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from micsa_workloads import CONFIGS  # noqa: E402

CFG = CONFIGS[4]
SWEEPS_PER_STEP = CFG.refresh_intervals[0]          # refresh every 10 sweeps
T_RUN = CFG.temperatures[0]
METRIC = "spin-flip attempts/ns (refresh + 10 sweeps + measure per step)"
UNIT = "attempts/ns"
# the microarchitecture guide's full-chip L2 throughput cap: ~6300 B/clk at the SM clock
L2_CAP_BYTES_PER_CLK = 6300.0
NCU_CSV = ROOT / "profiles" / "r2_ncu_metrics.csv"


def ncu_metrics(kernel_prefix, workload, capture="single pass"):
    """Per-launch counters of an ncu capture, from the committed summary profiles/r2_ncu_metrics.csv (columns: kernel,
    workload, metric, value in bytes / ns / counts, capture, commit; the commands are in profiles/r2_ncu_metrics.md).
    `capture` selects the rows whose capture column contains it.  Returns ({metric: value}, commit) or ({}, None)."""
    if not NCU_CSV.exists():
        return {}, None
    out, commit = {}, None
    with open(NCU_CSV) as f:
        for row in csv.DictReader(f):
            if row["kernel"].startswith(kernel_prefix) and row["workload"] == workload and capture in row["capture"]:
                out[row["metric"]] = float(row["value"])
                commit = row["commit"]
    return out, commit


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons during the timed region, sampled through
    NVML in-process every 2 ms (spawning nvidia-smi from a thread steals the
    launching thread's CPU and shows up as GPU idle time in a 0.3 ms step);
    falls back to nvidia-smi when the NVML binding is missing."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            # NVML indices follow the PCI order; honour CUDA_VISIBLE_DEVICES when it is a plain list
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            ids = [int(x) for x in vis.split(",")] if vis and all(x.strip().isdigit() for x in vis.split(",")) else None
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(ids[index] if ids else index)
            self.nvml = pynvml
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n = self.nvml
        sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
        r = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle)) \
            if hasattr(n, "nvmlDeviceGetCurrentClocksEventReasons") \
            else int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
        flags = [("hw_slowdown", 0x8), ("hw_thermal_slowdown", 0x40), ("sw_thermal_slowdown", 0x20),
                 ("sw_power_cap", 0x4)]
        self.rows.append([str(sm), str(self.sm_max)] + ["Active" if r & bit else "Not Active" for _, bit in flags])

    def run(self):
        while not self._stop_evt.is_set() and not os.environ.get('MICSA_NO_SAMPLER'):
            try:
                if self.nvml is not None:
                    self._sample_nvml()
                else:
                    out = subprocess.run(
                        ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                         "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                    f = [x.strip() for x in out.strip().split(",")]
                    if len(f) >= 6:
                        self.rows.append(f)
            except Exception:
                pass
            self._stop_evt.wait(0.002 if self.nvml is not None else 0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows for i in range(4) if r[2 + i].lower() == "active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": reasons, "samples": len(self.rows),
                "source": "nvml" if self.nvml is not None else "nvidia-smi"}


def oracle_step_rate(n_samples, steps, warmup, threads=None):
    """The oracle, as it stands, on the host cores: the same step on the first n_samples samples of config 4.  Its
    OpenMP loop spreads SYSTEMS over threads (oracle/micsa_oracle.c), so n_samples * n_replicas systems keep at most
    that many cores busy.  Returns (attempts/ns, threads busy, seconds)."""
    import oracle
    L, nr, seed = CFG.L, CFG.n_replicas, CFG.seed
    avail = os.cpu_count() or 1
    if threads is not None:
        oracle.set_num_threads(threads)
    else:
        oracle.set_num_threads(avail)
    busy = min(oracle.num_threads(), n_samples * nr)
    s = oracle.init_spins(L, n_samples, nr, seed)
    J = oracle.init_bonds(L, n_samples, seed)
    m = np.zeros_like(s, dtype=np.uint8)
    attempts = L ** 3 * n_samples * nr * SWEEPS_PER_STEP
    t_total = 0.0
    for k in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.refresh(L, m, seed, T_RUN, k)
        oracle.sweep(L, s, m, J, SWEEPS_PER_STEP)
        oracle.measure(L, s, m, J)
        if k >= warmup:
            t_total += time.perf_counter() - t0
    oracle.set_num_threads(avail)
    return attempts * steps / t_total / 1e9, busy, t_total


def oracle_sample_size():
    """Samples of config 4 the oracle legs run: one system per host core (2 replicas per sample)."""
    cores = os.cpu_count() or 1
    return max(1, min(CFG.n_samples, cores // CFG.n_replicas)), cores


def cpu_baseline_record(steps=1):
    n_s, cores = oracle_sample_size()
    rate_all, busy, secs = oracle_step_rate(n_s, steps, 0)
    rate_1, _, secs1 = oracle_step_rate(1, 1, 0, threads=1)
    rate_1 /= 1.0                                        # 2 systems, one thread
    return {"value": rate_all, "unit": UNIT, "cores": busy, "kind": "oracle",
            "host_cores": cores, "value_allcores": rate_all, "cores_used": busy,
            "value_1core": rate_1,
            "sample": f"{steps} step(s) (refresh + {SWEEPS_PER_STEP} sweeps + measure) of config 4 restricted to its "
                      f"first {n_s} samples x {CFG.n_replicas} replicas at L={CFG.L} = {n_s * CFG.n_replicas} systems, "
                      f"one OpenMP thread per system ({secs:.1f} s); value_1core: the first sample's 2 systems on "
                      f"one thread ({secs1:.1f} s)"}


def hbm_resident_record(micsa, tuned, stream, local_rank, rank, world, barrier, max_over_ranks, peak, e0, e1, kname):
    """The same kernels on a state larger than L2: 160^3 x 128 systems (the shape of the paper's timing table,
    PAPER.md:341-350), sweeps only and whole steps; frac = 7.5 bits per attempt over time against the HBM copy peak."""
    import torch
    from paper_2506_16240_b200.sharding import sample_offset
    L, nr, ns_big = CFG.L, CFG.n_replicas, 64
    sched_step = (T_RUN, SWEEPS_PER_STEP, SWEEPS_PER_STEP)
    gb = tuned(micsa.MicSA(L, ns_big, nr, CFG.seed, sample_offset=sample_offset(rank, ns_big), device=local_rank,
                           stream=stream))
    big = gb.layout_info()
    att_sweep = L ** 3 * ns_big * nr
    hbm = {"workload": f"table3_L{L}_{ns_big}x{nr}", "state_bytes": big["state_bytes"],
           "algorithmic_bytes_per_sweep": big["compulsory_bytes_per_sweep"], "peak": peak, "unit": "GB/s"}
    gb.refresh_demons(T_RUN, 0)
    for l2g in (0, 1):
        gb.set_tuning("l2_groups", l2g)
        gb.sweep(10)
        barrier()
        reps = []
        for _ in range(3):
            e0.record(stream); gb.sweep(10); e1.record(stream)
            torch.cuda.synchronize()
            reps.append(e0.elapsed_time(e1) / 10.0)
        ms = max_over_ranks(float(np.median(reps)))
        gbs = big["compulsory_bytes_per_sweep"] / (ms * 1e-3) / 1e9
        hbm[f"l2_groups_{l2g}"] = {"us_per_sweep": ms * 1e3, "attempts_per_ns": att_sweep * world / (ms * 1e6),
                                   "achieved": gbs, "frac": gbs / peak}
    gb.set_tuning("l2_groups", 1)
    gb.anneal([sched_step] * 20, step0=1)
    reps = []
    for rep in range(3):
        barrier()
        e0.record(stream); gb.anneal([sched_step] * 20, step0=21 + 20 * rep); e1.record(stream)
        barrier()
        reps.append(max_over_ranks(e0.elapsed_time(e1)))
    hbm["whole_step_attempts_per_ns"] = att_sweep * SWEEPS_PER_STEP * 20 * world / (float(np.median(reps)) * 1e6)
    hbm["whole_step_ms_repetitions"] = [t / 20 for t in reps]
    nb, nb_commit = ncu_metrics(kname, hbm["workload"])
    if "dram__bytes_read.sum" in nb:
        hbm["traffic_per_half_sweep"] = nb["dram__bytes_read.sum"] + nb.get("dram__bytes_write.sum", 0.0)
        hbm["traffic_source"] = f"{NCU_CSV.name} @ {nb_commit}"
    hbm["note"] = ("sweeps only, 10 per call; l2_groups_0 = every half-sweep over all 4 word lattices (each launch "
                   "streams the state through HBM), l2_groups_1 = the 10 sweeps lattice group by lattice group; "
                   "frac = 7.5 bits/attempt over time against the measured HBM copy peak")
    gb.destroy()
    return hbm


def gauss_record(micsa, stream, rank, world, barrier, max_over_ranks, peak, e0, e1):
    """SURVEY.md 8(f) rank 4, sub-record: continuous walkers with Gaussian couplings (Appendix C step 1),
    64^3 sites x 64 systems, float64: per EMCS one refresh from Eq. (9) and 10 x (sweep + forward-X wandering).
    Algorithmic bytes per attempt (one pass per sweep): n 8 r + 8 w, spin 1 r + 1 w (int8), bonds 3 x 8 B per site
    and sample read once per sweep and shared by the replicas = 24 / n_replicas."""
    import torch
    from micsa_workloads import gaussian_couplings
    L, ns, nr, T, n_emcs = 64, 32, 2, 1.0, 20
    N = L ** 3
    g = micsa.GaussMicSA(L, ns, nr, 6, sample_offset=rank * ns, stream=stream)
    g.set_couplings(gaussian_couplings((ns, 3, N), 7 + rank))
    g.set_walkers(1, 0)
    for k in range(3):
        g.refresh(T, k); g.sweep(10)
    reps = []
    for rep in range(3):
        barrier()
        e0.record(stream)
        for k in range(n_emcs):
            g.refresh(T, 10 + rep * n_emcs + k); g.sweep(10)
        e1.record(stream)
        barrier()
        reps.append(max_over_ranks(e0.elapsed_time(e1)))
    ms = float(np.median(reps))
    attempts = 10 * n_emcs * N * ns * nr * world
    bytes_per_attempt = 16.0 + 2.0 + 24.0 / nr
    gbs = attempts * bytes_per_attempt / (ms * 1e-3) / 1e9
    g.destroy()
    return {"workload": f"gauss_L{L}_{ns}x{nr}", "dtype": "f64", "attempts_per_ns": attempts / (ms * 1e6),
            "ms_per_emcs": ms / n_emcs, "algorithmic_bytes_per_attempt": bytes_per_attempt,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak},
            "note": "whole EMCS (refresh + 10 sweeps + 10 wandering half-cycles), one thread per (site, system); "
                    "state 335 MB, larger than L2"}


def run_reference(args, rank):
    if rank != 0:
        return
    n_s, cores = oracle_sample_size()
    rate, busy, secs = oracle_step_rate(n_s, args.steps, min(args.warmup, 1))
    sample = (f"config 4 restricted to its first {n_s} sample(s) x {CFG.n_replicas} replicas (L={CFG.L}), one OpenMP "
              f"thread per system on {cores} host cores; each step = refresh + {SWEEPS_PER_STEP} sweeps + measure")
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32",
        "data": "synthetic",
        "config": {"workload": CFG.name, "L": CFG.L, "n_samples": CFG.n_samples,
                   "n_replicas": CFG.n_replicas, "T": T_RUN, "sweeps_per_step": SWEEPS_PER_STEP},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": busy, "host_cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="micsa", choices=["micsa", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-hbm-resident", action="store_true")
    ap.add_argument("--only-hbm-resident", action="store_true",
                    help="profiling aid: run only the 160^3 x 128-system section (state larger than L2) and print it")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="micsa_set_tuning for A/B runs, e.g. --tune sweep_kernel=2")
    ap.add_argument("--walkers", action="store_true",
                    help="one forward-X walker per spin instead of a daemon (PAPER.md Sec. 2.6): every sweep is "
                         "followed by a wandering half-cycle; reported under its own metric name")
    ap.add_argument("--no-fuse-measure", action="store_true",
                    help="A/B: separate measurement kernel instead of counting inside the last sweep")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "micsa" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2506_16240_b200.build import build as build_lib
    if rank == 0:
        build_lib()
    import paper_2506_16240_b200 as micsa

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the MicSA library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        t = torch.tensor([x], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    L, ns, nr = CFG.L, CFG.n_samples, CFG.n_replicas
    # a high-priority stream for the path, so that the refresh prefetched on the
    # library's side stream only fills what the sweeps leave idle
    stream = torch.cuda.Stream(device=dev, priority=-1)
    torch.cuda.set_stream(stream)
    from paper_2506_16240_b200.sharding import sample_offset

    def tuned(g):
        if args.no_fuse_measure:
            g.set_tuning("fuse_measure", 0)
        if args.walkers:
            g.set_walkers(1)
        for kv in args.tune:
            k, v = kv.split("=")
            g.set_tuning(k, int(v))
        return g

    if args.only_hbm_resident:
        peak, _ = measured_peaks()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        hbm = hbm_resident_record(micsa, tuned, stream, local_rank, rank, world, barrier, max_over_ranks, peak, e0, e1,
                                  "half_sweep_pipe_kernel")
        if rank == 0:
            print(json.dumps({"hbm_resident": hbm}), flush=True)
        return

    g = tuned(micsa.MicSA(L, ns, nr, CFG.seed, sample_offset=sample_offset(rank, ns), device=local_rank,
                          stream=stream))
    info = g.layout_info()
    attempts_step = CFG.attempts_per_sweep * SWEEPS_PER_STEP
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    K, W = args.steps, args.warmup
    sched_step = (T_RUN, SWEEPS_PER_STEP, SWEEPS_PER_STEP)

    # ---- (1) l2_flushed: separately timed steps, closed window -------------------------------------------------
    # window of step k: [queue the generation of refresh k+1 on the side stream] [9 plain sweeps]
    # [measuring sweep, row D2H] [consume refresh k+1: wait for the side stream, swap the planes]
    def step(k, ev=None):
        if ev:
            ev[0].record(stream)
        g.prefetch_refresh(T_RUN, k + 1)
        if ev:
            ev[1].record(stream)
        g.sweep(SWEEPS_PER_STEP - 1)            # 18 plain half-sweep launches: the roofline kernel
        if ev:
            ev[2].record(stream)
        g.sweep_measure(1)                      # the last sweep also counts E, E_daemon, q; row D2H queued
        g.refresh_demons(T_RUN, k + 1)          # the refresh the next step starts from
        if ev:
            ev[3].record(stream)
        return g.measure_end()                  # host waits for the row (after the timed region)

    g.refresh_demons(T_RUN, 0)
    for k in range(W):
        step(k)
    barrier()
    launches0 = g.layout_info()["launches"]
    calls0 = g.counters()["philox_calls"]
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    barrier()
    wall0 = time.perf_counter()
    for k in range(K):
        flush.zero_()                                   # evict the state from L2 (untimed; nothing else is queued)
        step(W + k, evs[k])
    barrier()
    wall = time.perf_counter() - wall0
    launches_flushed = g.layout_info()["launches"] - launches0
    philox_words = 4.0 * (g.counters()["philox_calls"] - calls0)
    t_flushed_ms = max_over_ranks(sum(e[0].elapsed_time(e[3]) for e in evs))
    t_sweep_ms = sum(e[1].elapsed_time(e[2]) for e in evs)
    t_sweep_ms_max = max_over_ranks(t_sweep_ms)
    value_flushed = attempts_step * K * world / (t_flushed_ms * 1e6)

    # ---- (2) back_to_back: the K steps in ONE micsa_anneal call, one event pair --------------------------------
    g.anneal([sched_step] * max(W, K), step0=W + K + 1)              # warm-up of this path (rows, trace buffer)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches1 = g.layout_info()["launches"]
    reps_b2b = []
    for rep in range(3):                                             # K steps each; the median repetition is reported
        barrier()
        e0.record(stream)
        out = g.anneal([sched_step] * K, step0=(2 + rep) * (W + K) + 1)
        e1.record(stream)
        barrier()
        reps_b2b.append(max_over_ranks(e0.elapsed_time(e1)))
    clocks = sampler.stop()
    launches_b2b = (g.layout_info()["launches"] - launches1) // 3
    t_b2b_ms = float(np.median(reps_b2b))
    value_b2b = attempts_step * K * world / (t_b2b_ms * 1e6)
    assert out["E"].shape[0] == K
    if value_b2b <= value_flushed:
        value, t_step_ms, which, launches = value_b2b, t_b2b_ms, "back_to_back", launches_b2b
    else:
        value, t_step_ms, which, launches = value_flushed, t_flushed_ms, "l2_flushed", launches_flushed

    # steady state, no flush, back-to-back sweeps only
    barrier()
    e0.record(stream); g.sweep(100); e1.record(stream)
    torch.cuda.synchronize()
    sweep_only = CFG.attempts_per_sweep * 100 / (e0.elapsed_time(e1) * 1e6)

    # ---- roofline of the dominant kernel (plain half-sweep), live from the flushed steps ------------------------
    peak, peak_src = measured_peaks()
    sm_mhz = clocks.get("sm_mhz") or 1965.0
    l2_cap_gbs = L2_CAP_BYTES_PER_CLK * sm_mhz * 1e6 / 1e9
    n_launch = 2 * (SWEEPS_PER_STEP - 1) * K                 # the plain launches between events 1 and 2
    t_launch_s = t_sweep_ms * 1e-3 / n_launch
    alg_bytes = info["compulsory_bytes_per_sweep"] / 2          # per half-sweep launch
    achieved = alg_bytes / t_launch_s / 1e9
    kname = g.sweep_kernel_name() if hasattr(g, "sweep_kernel_name") else "half_sweep_pipe_kernel"
    ncu, ncu_commit = ncu_metrics(kname, CFG.name)
    traffic = None
    if "dram__bytes_read.sum" in ncu:
        traffic = ncu["dram__bytes_read.sum"] + ncu.get("dram__bytes_write.sum", 0.0)
    cold, _ = ncu_metrics(kname, CFG.name, capture="caches flushed")
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic,
                "traffic_source": f"{NCU_CSV.name} @ {ncu_commit}: dram__bytes_read.sum + dram__bytes_write.sum per launch, "
                                  "single-pass ncu of this command (L2 as the run leaves it)" if ncu else None,
                "traffic_cold": (cold["dram__bytes_read.sum"] + cold.get("dram__bytes_write.sum", 0.0))
                                if "dram__bytes_read.sum" in cold else None,
                "kernel": kname, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes,
                "us_per_launch": t_launch_s * 1e6,
                "convention": "compulsory one-pass traffic: 7.5 bits/attempt (spin 1r+1w, daemon 2r+2w, "
                              "bonds 1.5r shared by the replica pair)",
                "real_bound": "L2 <-> SM path: the 73.7 MB state of config 4 is L2-resident after the first sweep of a "
                              "step, DRAM traffic is ~0 warm; see l2_path and hbm_resident",
                "sweep_share_of_step": t_sweep_ms_max / t_flushed_ms,
                "note": "share = the 18 plain half-sweep launches of an l2_flushed step; the 2 launches of the last "
                        "sweep also do the measurement and are timed with the rest of the step"}
    if "lts__t_sectors_srcunit_tex.sum" in ncu:
        l2b = ncu["lts__t_sectors_srcunit_tex.sum"] * 32.0
        roofline["l2_path"] = {"bytes_per_launch": l2b, "achieved_gbs": l2b / t_launch_s / 1e9, "cap_gbs": l2_cap_gbs,
                               "frac": l2b / t_launch_s / 1e9 / l2_cap_gbs, "source": f"{NCU_CSV.name} @ {ncu_commit}",
                               "note": "secondary roofline: L2 <-> SM bytes of the ncu capture over the live launch "
                                       "time, against the guide's full-chip L2 throughput cap (6300 B/clk)"}

    # ---- end to end through the C ABI with host buffers ---------------------------------------------------------
    e2e = None
    if not args.no_e2e:
        s_host = torch.from_numpy(g.get_state(daemons=False, couplings=False)[0]).pin_memory()
        J_host = torch.from_numpy(g.get_state(spins=False, daemons=False)[2]).pin_memory()
        s_np, J_np = s_host.numpy(), J_host.numpy()
        n_run = max(K, 100)
        barrier()
        t0 = time.perf_counter()
        g.set_couplings(J_np)
        g.set_spins(s_np)
        out = g.anneal([sched_step] * n_run, step0=5000)
        barrier()
        dt = max_over_ranks(time.perf_counter() - t0)
        row_bytes = (2 * g.n_sys + g.n_pairs) * 8
        h2d = (s_np.nbytes + J_np.nbytes) / n_run + 16
        d2h = row_bytes + g.n_sys * 8 / n_run
        # the upload-every-step figure of round 1 (PCIe-bound by the one-byte-per-spin boundary layout)
        n_up = 3
        barrier()
        t1 = time.perf_counter()
        for k in range(n_up):
            g.set_couplings(J_np)
            g.set_spins(s_np)
            g.anneal([sched_step], step0=6000 + k)
        barrier()
        dt_up = max_over_ranks(time.perf_counter() - t1)
        # one host call per step, state left on the device
        n_res = max(20, K)
        barrier()
        t2 = time.perf_counter()
        for k in range(n_res):
            g.anneal([sched_step], step0=7000 + k)
        barrier()
        dt_res = max_over_ranks(time.perf_counter() - t2)
        e2e = {"value": attempts_step * n_run * world / (dt * 1e9), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_run,
               "what": f"wall clock of: micsa_set_couplings + micsa_set_spins from pinned host int8 arrays (one byte "
                       f"per spin / bond, {s_np.nbytes + J_np.nbytes} B once), micsa_anneal of {n_run} steps "
                       f"(refresh + 10 sweeps + measure each), measurement rows and min energies copied back",
               "upload_every_step": {"value": attempts_step * n_up * world / (dt_up * 1e9), "unit": UNIT,
                                     "h2d_bytes_per_step": s_np.nbytes + J_np.nbytes + 16,
                                     "d2h_bytes_per_step": row_bytes + g.n_sys * 8, "steps": n_up},
               "one_call_per_step": {"value": attempts_step * n_res * world / (dt_res * 1e9), "unit": UNIT,
                                     "h2d_bytes_per_step": 16, "d2h_bytes_per_step": row_bytes + g.n_sys * 8,
                                     "steps": n_res}}
    g.destroy()
    del flush

    hbm = None
    if not args.no_hbm_resident and not args.walkers:
        hbm = hbm_resident_record(micsa, tuned, stream, local_rank, rank, world, barrier, max_over_ranks, peak, e0, e1, kname)

    gauss = None
    if not args.no_hbm_resident and not args.walkers:
        gauss = gauss_record(micsa, stream, rank, world, barrier, max_over_ranks, peak, e0, e1)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_record()

    if rank == 0:
        line = {
            "metric": METRIC + (" [gamma=1 forward-X walkers]" if args.walkers else ""),
            "value": value, "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": t_step_ms / K, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": CFG.name, "L": L, "n_samples": ns, "n_replicas": nr, "T": T_RUN,
                       "sweeps_per_step": SWEEPS_PER_STEP, "state_bytes": info["state_bytes"],
                       "l2": "value = the lower of back_to_back (no flush: the 73.7 MB state is L2-resident in any "
                             "long run) and l2_flushed (256 MiB write between separately timed steps); inputs larger "
                             "than L2: see hbm_resident",
                       "sharding": "samples by rank, global sample offsets, no collective"},
            "value_is": which,
            "value_back_to_back": value_b2b, "ms_per_step_back_to_back": t_b2b_ms / K,
            "ms_per_step_back_to_back_repetitions": [t / K for t in reps_b2b],
            "value_l2_flushed": value_flushed, "ms_per_step_l2_flushed": t_flushed_ms / K,
            "rns_per_attempt": 1.0 / SWEEPS_PER_STEP,
            "philox_words_generated_per_attempt": philox_words / (attempts_step * K),
            "sweep_only_attempts_per_ns": sweep_only,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "hbm_resident": hbm, "continuous_daemons": gauss, "cpu_baseline": cpu, "wall_s": wall,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
