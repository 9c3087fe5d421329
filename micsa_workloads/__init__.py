"""Seeded synthetic workloads shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: only shapes, seeds,
temperature schedules and plain numpy random +-1 arrays.  Both the CUDA
library (through its Python binding) and the CPU oracle are fed from here.

The five configurations are BASELINE.json's `configs`, with the concrete
seeds / schedules fixed in DESIGN.md ("Input recipe").  The paper's workload
is itself synthetic (couplings +-1 with probability 1/2; fully
disordered start); its one real data set (the authors' L=160
sample and the Janus II trajectories) is not available and is stood in for by
seeded random samples of the same shape.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    n_samples: int
    n_replicas: int
    seed: int
    temperatures: tuple          # isothermal runs (one schedule per T) or ramp ends
    n_sweeps: int
    refresh_intervals: tuple     # sweeps between refreshes
    ramp_steps: int = 0          # >0: linear ramp T[0] -> T[1] in this many steps
    note: str = ""

    @property
    def N(self) -> int:
        return self.L ** 3

    @property
    def n_sys(self) -> int:
        return self.n_samples * self.n_replicas

    @property
    def attempts_per_sweep(self) -> int:
        return self.N * self.n_sys


CONFIGS = {
    1: Config("cfg1_L8_1x2", 8, 1, 2, 1, (2.0,), 1000, (10,),
              note="correctness config; measure every sweep"),
    2: Config("cfg2_L32_64x2", 32, 64, 2, 2, (3.0, 2.0, 1.5), 10_000, (10,),
              note="paramagnetic; <e> vs Metropolis"),
    3: Config("cfg3_L80_128x2", 80, 128, 2, 3, (0.7,), 100_000, (1, 10, 100),
              note="quench below T_c; refresh interval swept"),
    4: Config("cfg4_L160_16x2", 160, 16, 2, 4, (0.9,), 100_000, (10,),
              note="bandwidth-roofline headline"),
    5: Config("cfg5_L64_1024x1", 64, 1024, 1, 5, (3.0, 0.2), 10_000, (10,),
              ramp_steps=1000, note="annealing as optimisation"),
}


def fixed_interval_schedule(T, n_sweeps, interval, measure_every=0):
    """Configs 1-4: a demon refresh before sweep t whenever t % interval == 0
    (first refresh at t = 0; reading R3).  One schedule step =
    (T, n_sweeps_in_step, measure_every)."""
    if n_sweeps % interval:
        raise ValueError("n_sweeps must be a multiple of the refresh interval")
    return [(float(T), int(interval), int(measure_every))] * (n_sweeps // interval)


def linear_ramp_schedule(T_hi, T_lo, n_steps, sweeps_per_step, measure_every=None):
    """Config 5 (reading R12): T_k = T_hi - (T_hi - T_lo) k/(K-1),
    a refresh at every T step, measurement at the end of each step."""
    if measure_every is None:
        measure_every = sweeps_per_step
    if n_steps == 1:
        return [(float(T_hi), int(sweeps_per_step), int(measure_every))]
    return [(float(T_hi - (T_hi - T_lo) * k / (n_steps - 1)), int(sweeps_per_step),
             int(measure_every)) for k in range(n_steps)]


def schedule_for(cfg: Config, T=None, interval=None, n_sweeps=None, measure_every=0):
    """The schedule a BASELINE config runs (optionally truncated to n_sweeps)."""
    n = cfg.n_sweeps if n_sweeps is None else n_sweeps
    if cfg.ramp_steps:
        per = cfg.n_sweeps // cfg.ramp_steps
        full = linear_ramp_schedule(cfg.temperatures[0], cfg.temperatures[1],
                                    cfg.ramp_steps, per, measure_every or per)
        return full[: max(1, n // per)]
    T = cfg.temperatures[0] if T is None else T
    R = cfg.refresh_intervals[0] if interval is None else interval
    return fixed_interval_schedule(T, n, R, measure_every)


def pow2_schedule(T, s_max, measure_at_end=True):
    """The paper's own refresh rule (Sec. 2.8.1): refresh at
    t_s = 2^s, i.e. step s = refresh then 2^s timesteps, s = 0 .. s_max; one
    measurement at the end of every step."""
    return [(float(T), 1 << s, (1 << s) if measure_at_end else 0) for s in range(int(s_max) + 1)]


def random_pm1(shape, seed) -> np.ndarray:
    """i.i.d. fair +-1 int8 array (numpy PCG64) for tests that inject state
    through set_spins / set_couplings instead of the built-in Philox init."""
    rng = np.random.default_rng(seed)
    return (2 * rng.integers(0, 2, size=shape, dtype=np.int8) - 1).astype(np.int8)


def random_levels(shape, seed) -> np.ndarray:
    """i.i.d. uniform demon levels 0..3 (uint8) for state-injection tests."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, 4, size=shape, dtype=np.uint8)


def gaussian_couplings(shape, seed) -> np.ndarray:
    """i.i.d. N(0, 1) float64 couplings (numpy PCG64) for the continuous-daemon workload of the paper's Appendix C
    ("couplings are drawn from a Gaussian distribution J ~ N(0,1)").  Inputs only: both the CUDA
    library and the oracle receive the same array through their set-couplings calls."""
    return np.random.default_rng(seed).standard_normal(size=shape).astype(np.float64)
