#!/usr/bin/env python
"""bench.py -- MicSA hot-path throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl micsa|reference]

One STEP = one pass of the whole hot path over BASELINE
config 4 (L=160, 16 samples x 2 replicas, T=0.9): daemon refresh at T, then
10 checkerboard sweeps, then the E / E_daemon / q reductions.  Prints ONE JSON
line (rank 0).  `value` = spin-flip attempts per ns with the state resident in
HBM, timed with CUDA events on the library's stream, L2 flushed between steps;
the refresh of step k+1 is generated on the library's side stream during step
k (micsa_prefetch_refresh), so every timed step contains one generation;
`e2e` = the same step through the C ABI with HOST buffers (couplings + spins
uploaded from pinned host memory, observables read back) inside the timed
region.  N > 1: one process per GPU (torchrun), samples sharded by rank with
global sample offsets, no data-path collective (weak scaling).
"""
from __future__ import annotations

import argparse
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
# dram__bytes_read.sum + dram__bytes_write.sum per half-sweep launch from the
# ncu --set full capture summarised in profiles/r1c_final_launches_and_sweep.md
# (cold L2: ncu flushes caches before every replay; in a real step the 73.7 MB
# state stays in the 126 MB L2 after the first sweep)
NCU_TRAFFIC_BYTES_PER_LAUNCH = 57_401_600 + 172_288
# lts__t_sectors_srcunit_tex.sum * 32 B of the same capture: what crosses the L2 <-> SM path per launch -- the
# path that actually bounds the kernel (the state is L2-resident); the microarchitecture guide's full-chip L2
# throughput cap is ~6300 B/clk = 12.4 TB/s at 1.965 GHz
NCU_L2_BYTES_PER_LAUNCH = 3_355_957 * 32
L2_CAP_GBS = 6300 * 1.965


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


def oracle_step_rate(n_samples, steps, warmup):
    """The oracle, as it stands, on the host cores: same step on the first
    n_samples samples of config 4.  Returns (attempts/ns, cores, seconds)."""
    import oracle
    L, nr, seed = CFG.L, CFG.n_replicas, CFG.seed
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
    return attempts * steps / t_total / 1e9, oracle.num_threads(), t_total


def run_reference(args, rank):
    if rank != 0:
        return
    n_samples = 1                       # 2 systems of L=160: ~2-3 s of CPU work per step
    rate, cores, secs = oracle_step_rate(n_samples, args.steps, min(args.warmup, 1))
    sample = (f"config 4 restricted to its first {n_samples} sample(s) x {CFG.n_replicas} replicas "
              f"(L={CFG.L}); each step = refresh + {SWEEPS_PER_STEP} sweeps + measure")
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32",
        "data": "synthetic",
        "config": {"workload": CFG.name, "L": CFG.L, "n_samples": CFG.n_samples,
                   "n_replicas": CFG.n_replicas, "T": T_RUN, "sweeps_per_step": SWEEPS_PER_STEP},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
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
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="micsa_set_tuning for A/B runs, e.g. --tune pipe_smem_kb=48")
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
    g = micsa.MicSA(L, ns, nr, CFG.seed, sample_offset=sample_offset(rank, ns), device=local_rank,
                    stream=stream)
    if args.no_fuse_measure:
        g.set_tuning("fuse_measure", 0)
    if args.walkers:
        g.set_walkers(1)
    for kv in args.tune:
        k, v = kv.split("=")
        g.set_tuning(k, int(v))
    info = g.layout_info()
    attempts_step = CFG.attempts_per_sweep * SWEEPS_PER_STEP
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def step(k, ev=None):
        g.refresh_demons(T_RUN, k)              # consumes the planes prefetched during step k-1
        g.prefetch_refresh(T_RUN, k + 1)        # generated on the side stream under this step's sweeps
        if ev:
            ev[1].record(stream)
        g.sweep(SWEEPS_PER_STEP - 1)            # 18 plain half-sweep launches: the roofline kernel
        if ev:
            ev[2].record(stream)
        g.sweep_measure(1)                      # the last sweep also counts E, E_daemon, q; row D2H queued
        if ev:
            ev[3].record(stream)
        return g.measure_end()                  # host waits for the row (after the timed region)

    for k in range(args.warmup):
        step(k)
    barrier()
    launches0 = g.layout_info()["launches"]
    calls0 = g.counters()["philox_calls"]
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    barrier()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                                   # evict the state from L2 (untimed)
        ev = evs[k]
        ev[0].record(stream)
        step(args.warmup + k, ev)
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    launches = g.layout_info()["launches"] - launches0
    philox_words = 4.0 * (g.counters()["philox_calls"] - calls0)
    t_step_ms = sum(e[0].elapsed_time(e[3]) for e in evs)
    t_sweep_ms = sum(e[1].elapsed_time(e[2]) for e in evs)
    t_step_ms = max_over_ranks(t_step_ms)
    t_sweep_ms_max = max_over_ranks(t_sweep_ms)
    value = attempts_step * args.steps * world / (t_step_ms * 1e6)

    # steady state, no flush, back-to-back sweeps only (what a long run looks like)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream); g.sweep(100); e1.record(stream)
    torch.cuda.synchronize()
    sweep_only = CFG.attempts_per_sweep * 100 / (e0.elapsed_time(e1) * 1e6)

    # roofline of the dominant kernel (half-sweep), live from the timed region
    peak, peak_src = measured_peaks()
    n_launch = 2 * (SWEEPS_PER_STEP - 1) * args.steps        # the plain launches between events 1 and 2
    t_launch_s = t_sweep_ms * 1e-3 / n_launch
    alg_bytes = info["compulsory_bytes_per_sweep"] / 2          # per half-sweep launch
    achieved = alg_bytes / t_launch_s / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH,
                "kernel": "half_sweep_pipe_kernel<2,4,4>", "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes,
                "us_per_launch": t_launch_s * 1e6,
                "convention": "compulsory one-pass traffic: 7.5 bits/attempt (spin 1r+1w, daemon 2r+2w, "
                              "bonds 1.5r shared by the replica pair)",
                "l2_path": {"bytes_per_launch": NCU_L2_BYTES_PER_LAUNCH,
                            "achieved_gbs": NCU_L2_BYTES_PER_LAUNCH / t_launch_s / 1e9, "cap_gbs": L2_CAP_GBS,
                            "frac": NCU_L2_BYTES_PER_LAUNCH / t_launch_s / 1e9 / L2_CAP_GBS,
                            "note": "secondary roofline: L2 <-> SM bytes of the ncu capture over the live launch "
                                    "time, against the guide's full-chip L2 throughput cap"},
                "sweep_share_of_step": t_sweep_ms_max / t_step_ms,
                "note": "share = the 18 plain half-sweep launches of a step; the 2 launches of the last sweep "
                        "also do the measurement and are timed with the rest of the step"}

    # end to end through the C ABI with host buffers
    e2e = None
    if not args.no_e2e:
        s_host = torch.from_numpy(g.get_state(daemons=False, couplings=False)[0]).pin_memory()
        J_host = torch.from_numpy(g.get_state(spins=False, daemons=False)[2]).pin_memory()
        s_np, J_np = s_host.numpy(), J_host.numpy()
        n_e2e = max(3, min(args.steps, 5))
        barrier()
        t0 = time.perf_counter()
        for k in range(n_e2e):
            g.set_couplings(J_np)
            g.set_spins(s_np)
            out = g.anneal([(T_RUN, SWEEPS_PER_STEP, SWEEPS_PER_STEP)], step0=1000 + k)
        barrier()
        dt = max_over_ranks(time.perf_counter() - t0)
        h2d = s_np.nbytes + J_np.nbytes + 16
        d2h = (2 * g.n_sys + g.n_pairs + g.n_sys) * 8
        # the same host call with the state left on the device between steps (what a long run does:
        # the only per-step input is the 16-byte schedule entry, the output the measurement row)
        n_res = max(20, args.steps)
        barrier()
        t1 = time.perf_counter()
        for k in range(n_res):
            out = g.anneal([(T_RUN, SWEEPS_PER_STEP, SWEEPS_PER_STEP)], step0=2000 + k)
        barrier()
        dt_res = max_over_ranks(time.perf_counter() - t1)
        e2e = {"value": attempts_step * n_e2e * world / (dt * 1e9), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": n_e2e,
               "what": "micsa_set_couplings + micsa_set_spins from pinned host int8 (one byte per spin / bond: "
                       "the canonical boundary layout), micsa_anneal (refresh + 10 sweeps + measure), rows copied "
                       "back; PCIe-bound by construction",
               "state_resident": {"value": attempts_step * n_res * world / (dt_res * 1e9), "unit": UNIT,
                                  "h2d_bytes_per_step": 16, "d2h_bytes_per_step": d2h, "steps": n_res,
                                  "what": "micsa_anneal of one schedule step per host call, state left on the "
                                          "device, wall clock including launch, synchronisation and row read-back"}}
    g.destroy()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_s = 2
        rate, cores, secs = oracle_step_rate(n_s, 1, 0)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"one step (refresh + {SWEEPS_PER_STEP} sweeps + measure) of config 4 restricted "
                         f"to its first {n_s} samples x {nr} replicas at L={L}; {secs:.1f} s"}

    if rank == 0:
        line = {
            "metric": METRIC + (" [gamma=1 forward-X walkers]" if args.walkers else ""),
            "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_step_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": CFG.name, "L": L, "n_samples": ns, "n_replicas": nr, "T": T_RUN,
                       "sweeps_per_step": SWEEPS_PER_STEP, "state_bytes": info["state_bytes"],
                       "l2": "flushed between timed steps (256 MiB write); state 73.7 MB < 126 MB L2",
                       "sharding": "samples by rank, global sample offsets, no collective"},
            "rns_per_attempt": 1.0 / SWEEPS_PER_STEP,
            "philox_words_generated_per_attempt": philox_words / (attempts_step * args.steps),
            "sweep_only_attempts_per_ns": sweep_only,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "cpu_baseline": cpu, "wall_s": wall,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
