"""CPU oracle for MicSA (arxiv/paper_2506_16240) -- TEST INFRASTRUCTURE ONLY.

Thin ctypes/numpy wrapper around ``micsa_oracle.c`` (the paper's algorithm
written out with serial loops) and ``metropolis_oracle.c`` (an independent
textbook Metropolis used only as a pin).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2506_16240_b200`` and neither imports the other.

Array conventions (the canonical unpacked layout of the C-ABI boundary):
  s  int8  [n_samples, n_replicas, N]   spins, values -1/+1
  m  uint8 [n_samples, n_replicas, N]   demon level, n = 4 m
  J  int8  [n_samples, 3, N]            bond site i -> i + d
  site i = x + L*(y + L*z)
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_BUILD = _HERE / "_build"
_LIB = None

_c_i8p = ctypes.POINTER(ctypes.c_int8)
_c_u8p = ctypes.POINTER(ctypes.c_uint8)
_c_i64p = ctypes.POINTER(ctypes.c_int64)
_c_u32p = ctypes.POINTER(ctypes.c_uint32)
_c_u64p = ctypes.POINTER(ctypes.c_uint64)
_c_f64p = ctypes.POINTER(ctypes.c_double)


def build(force: bool = False) -> Path:
    """Compile the oracle's C sources with gcc into oracle/_build/liboracle.so."""
    _BUILD.mkdir(exist_ok=True)
    so = _BUILD / "liboracle.so"
    srcs = [_HERE / "micsa_oracle.c", _HERE / "metropolis_oracle.c", _HERE / "gauss_oracle.c"]
    if (not force and so.exists()
            and all(so.stat().st_mtime >= p.stat().st_mtime for p in srcs)):
        return so
    tmp = _BUILD / f"liboracle.{os.getpid()}.tmp.so"
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp)] + \
          [str(p) for p in srcs] + ["-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, so)
    return so


def lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(str(build()))
        _LIB.oracle_thresholds.argtypes = [ctypes.c_double, _c_u64p]
        _LIB.oracle_thresholds.restype = ctypes.c_int
        _LIB.oracle_refresh.restype = ctypes.c_int
        _LIB.oracle_refresh_alpha.restype = ctypes.c_int
        _LIB.oracle_metropolis_thresholds.argtypes = [ctypes.c_double, _c_u64p]
        _LIB.oracle_metropolis_thresholds.restype = ctypes.c_int
        _LIB.oracle_metropolis_sweep.restype = ctypes.c_int
        _LIB.oracle_metropolis_half_sweep.restype = ctypes.c_int
        _LIB.oracle_refresh_uniform.restype = ctypes.c_uint32
        _LIB.oracle_num_threads.restype = ctypes.c_int
        _LIB.oracle_gauss_refresh.restype = ctypes.c_int
        _LIB.oracle_gauss_uniform.restype = ctypes.c_double
    return _LIB


def _p(a, typ):
    return a.ctypes.data_as(typ)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(ctypes.c_int(n))


def philox4x32_10(ctr, key) -> np.ndarray:
    """One Philox4x32-10 block: ctr = 4 uint32, key = 2 uint32 -> 4 uint32."""
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    o = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_p(c, _c_u32p), _p(k, _c_u32p), _p(o, _c_u32p))
    return o


def init_spins(L, n_samples, n_replicas, seed, sample_offset=0) -> np.ndarray:
    N = L ** 3
    s = np.empty((n_samples, n_replicas, N), dtype=np.int8)
    lib().oracle_init_spins(ctypes.c_int(L), ctypes.c_int(n_samples),
                            ctypes.c_int(n_replicas), ctypes.c_uint64(seed),
                            ctypes.c_int(sample_offset), _p(s, _c_i8p))
    return s


def init_bonds(L, n_samples, seed, sample_offset=0) -> np.ndarray:
    N = L ** 3
    J = np.empty((n_samples, 3, N), dtype=np.int8)
    lib().oracle_init_bonds(ctypes.c_int(L), ctypes.c_int(n_samples),
                            ctypes.c_uint64(seed), ctypes.c_int(sample_offset),
                            _p(J, _c_i8p))
    return J


def _check(L, s, m, J):
    ns, nr, N = s.shape
    assert N == L ** 3 and s.dtype == np.int8 and s.flags.c_contiguous
    if m is not None:
        assert m.shape == s.shape and m.dtype == np.uint8 and m.flags.c_contiguous
    if J is not None:
        assert J.shape == (ns, 3, N) and J.dtype == np.int8 and J.flags.c_contiguous
    return ns, nr, N


def half_sweep(L, s, m, J, parity):
    """In-place half-sweep on sites of the given parity.
    Returns (accepted[n_sys], dE[n_sys]) as int64 arrays."""
    ns, nr, _ = _check(L, s, m, J)
    acc = np.zeros(ns * nr, dtype=np.int64)
    dE = np.zeros(ns * nr, dtype=np.int64)
    lib().oracle_half_sweep(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                            ctypes.c_int(parity), _p(s, _c_i8p), _p(m, _c_u8p),
                            _p(J, _c_i8p), _p(acc, _c_i64p), _p(dE, _c_i64p))
    return acc, dE


def sweep(L, s, m, J, n_sweeps=1) -> None:
    """n full sweeps, each = even half-sweep then odd half-sweep, in place."""
    ns, nr, _ = _check(L, s, m, J)
    lib().oracle_sweep(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                       ctypes.c_int(n_sweeps), _p(s, _c_i8p), _p(m, _c_u8p),
                       _p(J, _c_i8p))


def wander(L, m, axis=0, sign=+1, parity=0) -> None:
    """One half of the wandering cycle: walkers on sites of
    `parity` exchange with their neighbour along sign * axis, in place."""
    ns, nr, N = m.shape
    assert N == L ** 3 and m.dtype == np.uint8 and m.flags.c_contiguous
    assert axis in (0, 1, 2) and sign in (-1, 1) and parity in (0, 1)
    lib().oracle_wander(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), ctypes.c_int(axis),
                        ctypes.c_int(sign), ctypes.c_int(parity), _p(m, _c_u8p))


def timesteps_walkers(L, s, m, J, n_steps=1, t0=0) -> None:
    """n timesteps with one forward-X walker per spin:
    sweep, then the wandering half-cycle of parity t mod 2, t = t0, t0+1, ..."""
    ns, nr, _ = _check(L, s, m, J)
    lib().oracle_timesteps_walkers(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                                   ctypes.c_int(n_steps), ctypes.c_int64(t0),
                                   _p(s, _c_i8p), _p(m, _c_u8p), _p(J, _c_i8p))


def metropolis_thresholds(T: float) -> np.ndarray:
    """floor(exp(-4(k+1)/T) * 2^32), k = 0, 1, 2: acceptance thresholds for dH = 4, 8, 12."""
    thr = np.zeros(3, dtype=np.uint64)
    if lib().oracle_metropolis_thresholds(ctypes.c_double(T), _p(thr, _c_u64p)) != 0:
        raise ValueError(f"invalid temperature {T!r}")
    return thr


def metropolis_checkerboard(L, s, J, seed, T, tau0=0, n_sweeps=1, sample_offset=0, parity=None) -> None:
    """Standard Metropolis on the checkerboard with one Philox uniform per
    attempt, in place.  parity=None: n full sweeps with
    sweep indices tau0, tau0+1, ...; parity=0/1: one half-sweep with index tau0."""
    ns, nr, N = s.shape
    assert N == L ** 3 and s.dtype == np.int8 and s.flags.c_contiguous
    if parity is None:
        rc = lib().oracle_metropolis_sweep(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), ctypes.c_uint64(seed),
                                           ctypes.c_int(sample_offset), ctypes.c_double(T), ctypes.c_uint32(tau0),
                                           ctypes.c_int(n_sweeps), _p(s, _c_i8p), _p(J, _c_i8p))
    else:
        rc = lib().oracle_metropolis_half_sweep(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                                                ctypes.c_uint64(seed), ctypes.c_int(sample_offset),
                                                ctypes.c_double(T), ctypes.c_uint32(tau0), ctypes.c_int(parity),
                                                _p(s, _c_i8p), _p(J, _c_i8p))
    if rc != 0:
        raise ValueError(f"invalid temperature {T!r}")


def thresholds(T: float) -> np.ndarray:
    """Integer thresholds of the cumulative Eq. (11) (R7)."""
    thr = np.zeros(3, dtype=np.uint64)
    rc = lib().oracle_thresholds(ctypes.c_double(T), _p(thr, _c_u64p))
    if rc != 0:
        raise ValueError(f"invalid temperature {T!r}")
    return thr


def refresh(L, m, seed, T, step, sample_offset=0) -> None:
    """Overwrite every demon with a draw from Eq. (11) at temperature T."""
    ns, nr, N = m.shape
    assert N == L ** 3 and m.dtype == np.uint8 and m.flags.c_contiguous
    rc = lib().oracle_refresh(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                              ctypes.c_uint64(seed), ctypes.c_int(sample_offset),
                              ctypes.c_double(T), ctypes.c_uint32(step),
                              _p(m, _c_u8p))
    if rc != 0:
        raise ValueError(f"invalid temperature {T!r}")


def refresh_alpha(L, m, seed, T, step, alpha, sample_offset=0) -> None:
    """Refresh of the alpha-th daemon family (gamma daemons per spin)."""
    ns, nr, N = m.shape
    assert N == L ** 3 and m.dtype == np.uint8 and m.flags.c_contiguous
    rc = lib().oracle_refresh_alpha(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                                    ctypes.c_uint64(seed), ctypes.c_int(sample_offset),
                                    ctypes.c_double(T), ctypes.c_uint32(step), ctypes.c_int(alpha),
                                    _p(m, _c_u8p))
    if rc != 0:
        raise ValueError(f"invalid temperature {T!r} or alpha {alpha!r}")


def refresh_uniform(i, g, rep, step, seed) -> int:
    """The 32-bit uniform of the demon at site i of global sample g, replica
    rep, refresh index step (R8)."""
    return int(lib().oracle_refresh_uniform(ctypes.c_uint32(i), ctypes.c_uint32(g),
                                            ctypes.c_uint32(rep), ctypes.c_uint32(step),
                                            ctypes.c_uint64(seed)))


def measure(L, s, m, J):
    """Exact integer sums: E[n_sys], Edem[n_sys], Q[n_samples*nr(nr-1)/2]."""
    ns, nr, _ = _check(L, s, m, J)
    E = np.zeros(ns * nr, dtype=np.int64)
    Ed = np.zeros(ns * nr, dtype=np.int64)
    Q = np.zeros(ns * nr * (nr - 1) // 2, dtype=np.int64)
    lib().oracle_measure(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                         _p(s, _c_i8p), _p(m, _c_u8p), _p(J, _c_i8p),
                         _p(E, _c_i64p), _p(Ed, _c_i64p),
                         _p(Q, _c_i64p) if Q.size else None)
    return E, Ed, Q


def c4(L, s) -> np.ndarray:
    """S[pair, axis, r] = sum_x q_x q_{x + r e_axis}, q = s^a s^b, r = 0..L/2 (Eq. 16
    before normalisation); pairs ordered like Q in measure()."""
    ns, nr, N = s.shape
    assert N == L ** 3 and s.dtype == np.int8 and s.flags.c_contiguous
    S = np.zeros((ns * nr * (nr - 1) // 2, 3, L // 2 + 1), dtype=np.int64)
    lib().oracle_c4(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), _p(s, _c_i8p), _p(S, _c_i64p))
    return S


def c4_normalised(L, S) -> np.ndarray:
    """Eq. (16) with its normalisation: C4(r) of ONE sample from the sums of all its replica pairs,
    S[pairs_of_the_sample, axis, r] -> sum over pairs and axes / (3 N N_R (N_R - 1) / 2) = mean over pairs and axes / N."""
    S = np.asarray(S, dtype=np.float64)
    return S.sum(axis=(0, 1)) / (3.0 * S.shape[0] * L ** 3)


def xi(C4, c_min=0.0):
    """Eq. (17)-(18) on the lattice, reading R22 of DESIGN.md (the paper defers the technical details
    of estimating I_n to its refs. [61, 46]): C4 is known at r = 0, 1, ..., L/2; the integral over [0, r_cut] is taken
    with the trapezoidal rule, r_cut = the last r before C4 first drops to c_min or below (noise floor chosen by the
    caller, e.g. three times the sample error), no tail added.  Returns (I_1, I_2, I_3, xi_12 = I_2 / I_1,
    xi_23 / xi_12 = I_3 I_1 / I_2^2)."""
    C4 = np.asarray(C4, dtype=np.float64)
    below = np.nonzero(C4 <= c_min)[0]
    n = int(below[0]) if below.size else C4.size
    if n < 2:
        raise ValueError("C4 is at or below the cut-off from r = 1 on")
    r = np.arange(n, dtype=np.float64)
    I = [float(np.trapezoid(r ** k * C4[:n], r)) for k in (1, 2, 3)]
    return I[0], I[1], I[2], I[1] / I[0], (I[2] / I[1]) / (I[1] / I[0])


def metropolis(L, s, J, T, n_sweeps, seed):
    """Independent textbook Metropolis (metropolis_oracle.c); s updated in
    place; returns the energy per spin after each sweep, float64
    [n_sweeps, n_sys]."""
    ns, nr, N = _check(L, s, None, J)
    e = np.zeros((n_sweeps, ns * nr), dtype=np.float64)
    lib().metropolis_run(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr),
                         ctypes.c_double(T), ctypes.c_int(n_sweeps),
                         ctypes.c_uint64(seed), _p(s, _c_i8p), _p(J, _c_i8p),
                         _p(e, _c_f64p))
    return e


# ---------------------------------------------------------------- continuous daemons, Gaussian couplings
# (gauss_oracle.c; PAPER.md:136-140 Eq. 9, :436-454 Appendix C).  s int8 [ns, nr, N], n float64 [ns, nr, N],
# J float64 [ns, 3, N].
def _check_gauss(L, s, n, J):
    ns, nr, N = s.shape
    assert N == L ** 3 and s.dtype == np.int8 and s.flags.c_contiguous
    if n is not None:
        assert n.shape == s.shape and n.dtype == np.float64 and n.flags.c_contiguous
    if J is not None:
        assert J.shape == (ns, 3, N) and J.dtype == np.float64 and J.flags.c_contiguous
    return ns, nr


def gauss_refresh(L, n, seed, T, step, sample_offset=0) -> None:
    ns, nr, N = n.shape
    assert n.dtype == np.float64 and n.flags.c_contiguous and N == L ** 3
    rc = lib().oracle_gauss_refresh(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), ctypes.c_uint64(seed),
                                    ctypes.c_double(T), ctypes.c_uint32(step), ctypes.c_int(sample_offset),
                                    _p(n, _c_f64p))
    if rc != 0:
        raise ValueError("temperature must be finite and > 0")


def gauss_uniform(i, gsample, rep, step, seed) -> float:
    return float(lib().oracle_gauss_uniform(ctypes.c_int64(i), ctypes.c_int(gsample), ctypes.c_int(rep),
                                            ctypes.c_uint32(step), ctypes.c_uint64(seed)))


def gauss_half_sweep(L, s, n, J, parity) -> None:
    ns, nr = _check_gauss(L, s, n, J)
    lib().oracle_gauss_half_sweep(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), _p(s, _c_i8p),
                                  _p(n, _c_f64p), _p(J, _c_f64p), ctypes.c_int(parity))


def gauss_sweep(L, s, n, J, n_sweeps=1, walkers=False, t0=0) -> None:
    """n_sweeps timesteps: even half-sweep, odd half-sweep; with walkers the forward-X wandering
    half-cycle of parity t mod 2 follows every sweep (Appendix C step 1(b); R15)."""
    for k in range(n_sweeps):
        gauss_half_sweep(L, s, n, J, 0)
        gauss_half_sweep(L, s, n, J, 1)
        if walkers:
            gauss_wander(L, n, 0, +1, (t0 + k) & 1)


def gauss_wander(L, n, axis=0, sign=+1, parity=0) -> None:
    ns, nr, N = n.shape
    assert n.dtype == np.float64 and n.flags.c_contiguous
    lib().oracle_gauss_wander(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), _p(n, _c_f64p),
                              ctypes.c_int(axis), ctypes.c_int(sign), ctypes.c_int(parity))


def gauss_measure(L, s, n, J):
    ns, nr = _check_gauss(L, s, n, J)
    E = np.zeros(ns * nr, np.float64)
    Ed = np.zeros(ns * nr, np.float64)
    Q = np.zeros(ns * (nr * (nr - 1) // 2), np.int64)
    lib().oracle_gauss_measure(ctypes.c_int(L), ctypes.c_int(ns), ctypes.c_int(nr), _p(s, _c_i8p), _p(n, _c_f64p),
                               _p(J, _c_f64p), _p(E, _c_f64p), _p(Ed, _c_f64p), _p(Q, _c_i64p))
    return E, Ed, Q
