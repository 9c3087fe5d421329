"""Statistical / closed-form pins for the CPU oracle (-m "not gpu").

  P5  refresh histogram vs Eq. (11), mean vs Eq. (12)
  R7  integer thresholds: monotone, no 2^32 wrap, = Eq. (11) to 2^-32
  P7  2x2x2 lattice: long-run <e> == brute-force Boltzmann average (3 sigma)
  P8  high-T equilibrium <e> == independent Metropolis (3 sigma)
  P10 equilibrium demon energy before a refresh ~ Eq. (12)
"""
import itertools
import math

import numpy as np
import pytest

from micsa_workloads import random_pm1
from oracle import driver


def eq11(T):
    """p(n = 4m), m = 0..3, exactly as printed in PAPER.md:156 (Eq. 11)."""
    b = 1.0 / T
    return np.array([math.exp(-4 * m * b) * (1 - math.exp(-4 * b)) / (1 - math.exp(-16 * b))
                     for m in range(4)])


def eq12(T):
    """<H_aux>/(gamma N) exactly as printed in PAPER.md:186 (Eq. 12)."""
    b = 1.0 / T
    return (4 * math.exp(-4 * b) / (1 - math.exp(-4 * b))
            - 16 * math.exp(-16 * b) / (1 - math.exp(-16 * b)))


@pytest.mark.parametrize("T", [3.0, 2.0, 1.5, 0.9, 0.7, 0.2, 50.0])
def test_thresholds_match_eq11(oracle, T):
    thr = oracle.thresholds(T).astype(object)
    assert 0 < thr[0] <= thr[1] <= thr[2] <= 2 ** 32
    p = eq11(T)
    assert abs(p.sum() - 1) < 1e-14
    cdf = np.cumsum(p)[:3]
    for k in range(3):
        assert abs(int(thr[k]) / 2.0 ** 32 - cdf[k]) <= 2.0 ** -32 + 1e-15
    if T == 0.2:   # e^{-20} ~ 2e-9: levels 2, 3 have probability < 2^-32
        assert int(thr[1]) == 2 ** 32 and int(thr[2]) == 2 ** 32


@pytest.mark.parametrize("T", [-1.0, 0.0, float("nan"), float("inf")])
def test_thresholds_reject_bad_temperature(oracle, T):
    with pytest.raises(ValueError):
        oracle.thresholds(T)


@pytest.mark.parametrize("T", [3.0, 2.0, 1.5, 0.9])
def test_refresh_histogram_and_mean(oracle, T):
    L, ns, nr = 16, 5, 2
    N = L ** 3
    m = np.full((ns, nr, N), 7, dtype=np.uint8)
    oracle.refresh(L, m, seed=2024, T=T, step=3)
    assert m.max() <= 3
    n_tot = m.size
    counts = np.bincount(m.reshape(-1), minlength=4).astype(float)
    p = eq11(T)
    # every bin within 4.5 sigma of its binomial expectation
    for k in range(4):
        sig = math.sqrt(n_tot * p[k] * (1 - p[k]))
        assert abs(counts[k] - n_tot * p[k]) < 4.5 * sig + 1, (T, k)
    mean_n = 4.0 * m.astype(np.float64).mean()
    var_n = 16.0 * (np.arange(4) ** 2 * p).sum() - eq12(T) ** 2
    assert abs(mean_n - eq12(T)) < 4.5 * math.sqrt(var_n / n_tot)
    # per-system streams look independent: system means scatter like 1/sqrt(N)
    sys_means = 4.0 * m.reshape(ns * nr, N).mean(axis=1)
    assert np.all(np.abs(sys_means - eq12(T)) < 5 * math.sqrt(var_n / N))
    flat = m.reshape(ns * nr, N)
    assert len({flat[k].tobytes() for k in range(ns * nr)}) == ns * nr


def test_refresh_uniform_is_uniform_and_independent(oracle):
    """DESIGN.md R8: the bit-plane assembly must give one fair 32-bit integer
    per demon, independent between demons that share Philox calls (the 16
    samples of a block) and between sites / replicas / steps."""
    seed, n_sites = 77, 1500
    U = np.array([[oracle.refresh_uniform(i, g, 0, 4, seed) for g in range(32, 48)]
                  for i in range(n_sites)], dtype=np.uint64)          # one 16-sample block
    flat = U.reshape(-1).astype(np.float64) / 2.0 ** 32
    n = flat.size
    # Kolmogorov-Smirnov against U(0,1): D * sqrt(n) < 1.95  (p ~ 1e-3)
    srt = np.sort(flat)
    D = max(np.max(np.arange(1, n + 1) / n - srt), np.max(srt - np.arange(n) / n))
    assert D * math.sqrt(n) < 1.95
    # every one of the 32 bit positions is fair (5 sigma)
    for k in range(32):
        ones = int(((U >> np.uint64(k)) & np.uint64(1)).sum())
        assert abs(ones - n / 2) < 5 * math.sqrt(n / 4), k
    # demons sharing a block are uncorrelated and never share bits systematically
    Z = (U.astype(np.float64) / 2.0 ** 32 - 0.5) * math.sqrt(12.0)
    C = (Z.T @ Z) / n_sites
    off = C - np.diag(np.diag(C))
    assert np.max(np.abs(off)) < 5 / math.sqrt(n_sites)
    x = U[:, :-1] ^ U[:, 1:]                                         # neighbours differ in ~16 bits
    pop = np.array([bin(int(v)).count("1") for v in x.reshape(-1)])
    assert abs(pop.mean() - 16) < 5 * math.sqrt(8.0 / pop.size)
    assert len(set(U.reshape(-1).tolist())) > n - 4                  # no systematic collisions
    # replica, step and sample block all enter
    base = oracle.refresh_uniform(5, 33, 0, 4, seed)
    assert len({base, oracle.refresh_uniform(5, 33, 1, 4, seed), oracle.refresh_uniform(5, 33, 0, 5, seed),
                oracle.refresh_uniform(5, 49, 0, 4, seed), oracle.refresh_uniform(6, 33, 0, 4, seed),
                oracle.refresh_uniform(5, 33, 0, 4, seed + 1)}) == 6


def test_refresh_uniform_uses_every_philox_bit_once(oracle):
    """The 16 uniforms of a block are a bit-matrix transpose of the four Philox
    blocks (R8): same multiset of bits, plane k = 8c + 2j + h is the
    h-th 16-bit half of output word j of call c, most significant plane first."""
    seed, i, B, rep, step = 0xABCDEF12345, 1234, 7, 3, 99
    key = [seed & 0xFFFFFFFF, seed >> 32]
    words = np.concatenate([oracle.philox4x32_10([i, B | (c << 28), rep, step], key) for c in range(4)])
    halves = words.view(np.uint16)                                   # little endian: low half first
    planes = np.unpackbits(halves.view(np.uint8).reshape(32, 2), axis=1, bitorder="little")   # [plane, lane]
    for lane in range(16):
        u = int("".join(str(b) for b in planes[:, lane]), 2)
        assert u == oracle.refresh_uniform(i, 16 * B + lane, rep, step, seed)


def test_refresh_is_a_pure_function_of_its_counters(oracle):
    L, ns, nr = 4, 6, 2
    N = L ** 3
    a = np.zeros((ns, nr, N), dtype=np.uint8)
    b = np.full((ns, nr, N), 3, dtype=np.uint8)
    oracle.refresh(L, a, 9, 2.0, 5)
    oracle.refresh(L, b, 9, 2.0, 5)
    np.testing.assert_array_equal(a, b)             # old demons are thrown away
    c = np.zeros_like(a)
    oracle.refresh(L, c, 9, 2.0, 6)
    assert not np.array_equal(a, c)                 # step enters the counter
    d = np.zeros_like(a)
    oracle.refresh(L, d, 10, 2.0, 5)
    assert not np.array_equal(a, d)                 # seed is the key
    # sharding by sample: samples [4, 6) generated with sample_offset 4
    e = np.zeros((2, nr, N), dtype=np.uint8)
    oracle.refresh(L, e, 9, 2.0, 5, sample_offset=4)
    np.testing.assert_array_equal(e, a[4:6])
    # monotone coupling in T: same uniforms, higher T -> level never lower
    hot = np.zeros_like(a)
    oracle.refresh(L, hot, 9, 3.0, 5)
    assert np.all(hot >= a) and np.any(hot > a)


def test_init_is_fair_and_shardable(oracle):
    L, ns, nr = 8, 40, 2
    s = oracle.init_spins(L, ns, nr, seed=7)
    J = oracle.init_bonds(L, ns, seed=7)
    assert set(np.unique(s)) == {-1, 1} and set(np.unique(J)) == {-1, 1}
    for a in (s, J):
        n = a.size
        assert abs(a.astype(np.float64).sum()) < 4.5 * math.sqrt(n)
    # replicas, samples and directions are distinct streams
    flat = np.concatenate([s.reshape(ns * nr, -1), J.reshape(ns * 3, -1)])
    c = np.abs(flat.astype(np.float64) @ flat.T.astype(np.float64)) / flat.shape[1]
    np.fill_diagonal(c, 0)
    assert c.max() < 6 / math.sqrt(flat.shape[1])
    np.testing.assert_array_equal(oracle.init_spins(L, 8, nr, 7, sample_offset=32), s[32:40])
    np.testing.assert_array_equal(oracle.init_bonds(L, 8, 7, sample_offset=32), J[32:40])


# ---------------------------------------------------------------- P7 brute force
def _boltzmann_2x2x2(J, T):
    """Exact <e> of the 8-spin periodic cube with its 24 distinct bonds
    (R10), by enumeration of all 2^8 states; no oracle code."""
    L, N = 2, 8
    idx = lambda x, y, z: (x % L) + L * ((y % L) + L * (z % L))
    bonds = []
    for z, y, x in itertools.product(range(2), repeat=3):
        i = idx(x, y, z)
        bonds += [(i, idx(x + 1, y, z), J[0][i]), (i, idx(x, y + 1, z), J[1][i]),
                  (i, idx(x, y, z + 1), J[2][i])]
    assert len(bonds) == 24
    Z = 0.0
    Esum = 0.0
    for bits in range(256):
        s = [1 - 2 * ((bits >> k) & 1) for k in range(N)]
        E = -sum(j * s[a] * s[b] for a, b, j in bonds)
        w = math.exp(-E / T)
        Z += w
        Esum += E * w
    return Esum / Z / N


@pytest.mark.parametrize("T,seed", [(2.0, 11), (3.0, 12)])
def test_2x2x2_matches_exact_boltzmann(oracle, T, seed):
    L, N, nr = 2, 8, 64
    J = random_pm1((1, 3, N), seed)
    exact = _boltzmann_2x2x2(J[0].tolist(), T)
    s = oracle.init_spins(L, 1, nr, seed)
    m = np.zeros((1, nr, N), dtype=np.uint8)
    n_sweeps, therm = 6000, 200
    sched = [(T, 10, 1)] * (n_sweeps // 10)
    out = driver.anneal(L, s, m, J, seed, sched)
    e = out["E"][therm:] / float(N)                       # [t, replica]
    per_rep = e.mean(axis=0)                              # independent replicas
    mean, err = per_rep.mean(), per_rep.std(ddof=1) / math.sqrt(nr)
    assert err < 0.01
    assert abs(mean - exact) < 3 * err, (mean, exact, err)
    # and the demons sit at Eq. (12) just after... and on average before a refresh (P10)
    ed = out["Edem"][therm:][9::10] / float(N)            # last sweep before each refresh
    per_rep_d = ed.mean(axis=0)
    derr = per_rep_d.std(ddof=1) / math.sqrt(nr)
    assert abs(per_rep_d.mean() - eq12(T)) < 3 * derr + 1e-12, (per_rep_d.mean(), eq12(T), derr)


def test_2x2x2_wrong_physics_would_fail():
    """Sanity of the pin itself: the exact average separates T=2 from T=3 and a
    24-bond from a 12-bond cube by many sigma of the test above."""
    J = random_pm1((1, 3, 8), 11)[0].tolist()
    assert abs(_boltzmann_2x2x2(J, 2.0) - _boltzmann_2x2x2(J, 3.0)) > 0.1


# ---------------------------------------------------------------- P8 Metropolis
@pytest.mark.parametrize("T", [3.0, 2.0])
def test_equilibrium_energy_matches_metropolis(oracle, T):
    L, ns, nr = 6, 4, 8
    N = L ** 3
    J = oracle.init_bonds(L, ns, seed=21)
    s_mic = oracle.init_spins(L, ns, nr, seed=21)
    s_met = s_mic.copy()
    m = np.zeros((ns, nr, N), dtype=np.uint8)
    n_sweeps, therm = 3000, 500
    out = driver.anneal(L, s_mic, m, J, 21, [(T, 10, 1)] * (n_sweeps // 10))
    e_mic = (out["E"][therm:] / float(N)).mean(axis=0).reshape(ns, nr)
    e_met = oracle.metropolis(L, s_met, J, T, n_sweeps, seed=5)[therm:].mean(axis=0).reshape(ns, nr)
    # compare sample by sample (same couplings), error from replica scatter
    for k in range(ns):
        d = e_mic[k].mean() - e_met[k].mean()
        err = math.sqrt(e_mic[k].var(ddof=1) / nr + e_met[k].var(ddof=1) / nr)
        assert abs(d) < 3 * err + 1e-9, (T, k, d, err)
    d_all = e_mic.mean() - e_met.mean()
    err_all = math.sqrt(e_mic.var(ddof=1) / e_mic.size + e_met.var(ddof=1) / e_met.size)
    assert abs(d_all) < 3 * err_all
    # coarse textbook scale: e ~ -3 tanh(beta) to leading order at high T
    assert abs(e_mic.mean() / (-3 * math.tanh(1 / T)) - 1) < 0.12


def test_metropolis_oracle_itself_on_2x2x2(oracle):
    """The comparator is pinned too: Metropolis on the 8-spin cube == exact."""
    T, N, nr = 2.0, 8, 64
    J = random_pm1((1, 3, N), 33)
    exact = _boltzmann_2x2x2(J[0].tolist(), T)
    s = oracle.init_spins(2, 1, nr, 33)
    e = oracle.metropolis(2, s, J, T, 6000, seed=8)[200:]
    per_rep = e.mean(axis=0)
    err = per_rep.std(ddof=1) / math.sqrt(nr)
    assert abs(per_rep.mean() - exact) < 3 * err


# ---------------------------------------------------------------- walkers (Sec. 2.6, 2.8)
@pytest.mark.parametrize("L", [2, 4, 6])
@pytest.mark.parametrize("axis,sign", [(0, 1), (1, 1), (2, 1), (0, -1), (1, -1), (2, -1)])
def test_wandering_is_a_permutation_with_period_L(oracle, L, axis, sign):
    """after L/2 cycles (L timesteps) every walker is back where it
    started; each half-cycle is an exchange, hence its own inverse and a
    permutation; walkers starting on even sites travel one site per timestep
    in the wandering direction, the others against it."""
    ns, nr, N = 2, 2, L ** 3
    m0 = (np.arange(ns * nr * N, dtype=np.int64) % 251).astype(np.uint8).reshape(ns, nr, N)   # labels, not levels
    m = m0.copy()
    oracle.wander(L, m, axis, sign, 0); oracle.wander(L, m, axis, sign, 0)
    np.testing.assert_array_equal(m, m0)                                   # exchange twice = identity
    for t in range(L):
        oracle.wander(L, m, axis, sign, t & 1)
        assert sorted(m[1, 1].tolist()) == sorted(m0[1, 1].tolist())      # permutation
        if 0 < t + 1 < L and L > 2:
            assert not np.array_equal(m, m0)
    np.testing.assert_array_equal(m, m0)                                   # period L
    # direction: follow the walker that starts at the origin (an even site)
    if L >= 4:
        tag = np.zeros((1, 1, N), np.uint8); tag[0, 0, 0] = 1
        for t in range(L // 2):
            oracle.wander(L, tag, axis, sign, t & 1)
        pos = int(np.flatnonzero(tag[0, 0])[0])
        xyz = [pos % L, (pos // L) % L, pos // (L * L)]
        want = [0, 0, 0]; want[axis] = (sign * (L // 2)) % L
        assert xyz == want


def test_walkers_conserve_total_energy_and_do_not_touch_spins(oracle):
    L, ns, nr = 6, 3, 2
    N = L ** 3
    s, J = random_pm1((ns, nr, N), 61), random_pm1((ns, 3, N), 62)
    m = np.zeros((ns, nr, N), np.uint8)
    oracle.refresh(L, m, 5, 1.5, 0)
    E0, Ed0, _ = oracle.measure(L, s, m, J)
    s_before = s.copy()
    mw = m.copy()
    oracle.wander(L, mw, 0, +1, 0)
    assert not np.array_equal(mw, m)
    assert np.array_equal(oracle.measure(L, s, mw, J)[1], Ed0)             # walker energy only moves around
    for t in range(9):
        oracle.timesteps_walkers(L, s, m, J, 1, t0=t)
        E, Ed, _ = oracle.measure(L, s, m, J)
        np.testing.assert_array_equal(E + Ed, E0 + Ed0)
    # same thing in one call
    s2, m2 = s_before.copy(), np.zeros_like(m); oracle.refresh(L, m2, 5, 1.5, 0)
    oracle.timesteps_walkers(L, s2, m2, J, 9, t0=0)
    np.testing.assert_array_equal(s2, s); np.testing.assert_array_equal(m2, m)
    # and it differs from fixed daemons
    s3, m3 = s_before.copy(), np.zeros_like(m); oracle.refresh(L, m3, 5, 1.5, 0)
    oracle.sweep(L, s3, m3, J, 9)
    assert not np.array_equal(s3, s)


@pytest.mark.parametrize("T,seed", [(2.0, 21), (3.0, 22)])
def test_2x2x2_walkers_match_exact_boltzmann(oracle, T, seed):
    """Same pin as P7 with walkers: wandering must not spoil stationarity."""
    L, N, nr = 2, 8, 64
    J = random_pm1((1, 3, N), seed)
    exact = _boltzmann_2x2x2(J[0].tolist(), T)
    s = oracle.init_spins(L, 1, nr, seed)
    m = np.zeros((1, nr, N), dtype=np.uint8)
    n_sweeps, therm = 6000, 200
    sched = [(T, 10, 1)] * (n_sweeps // 10)
    out = driver.anneal(L, s, m, J, seed, sched, walkers=True)
    e = out["E"][therm:] / float(N)
    per_rep = e.mean(axis=0)
    mean, err = per_rep.mean(), per_rep.std(ddof=1) / math.sqrt(nr)
    assert err < 0.01
    assert abs(mean - exact) < 3 * err, (mean, exact, err)


# ---------------------------------------------------------------- canonical comparator
def test_checkerboard_metropolis_acceptance_rates(oracle):
    """Single-attempt pins: dH <= 0 always flips; dH = +12 / +8 / +4 flips with
    probability exp(-dH/T) (binomial, 4.5 sigma); thresholds = the Boltzmann
    factors to 2^-32."""
    T = 6.0
    thr = oracle.metropolis_thresholds(T).astype(object)
    for k in range(3):
        assert abs(int(thr[k]) / 2.0 ** 32 - math.exp(-4.0 * (k + 1) / T)) <= 2.0 ** -32 + 1e-15
    hot = [int(v) for v in oracle.metropolis_thresholds(1e9)]
    assert 2 ** 32 - 100 < hot[2] <= hot[1] <= hot[0] <= 2 ** 32
    with pytest.raises(ValueError):
        oracle.metropolis_thresholds(0.0)
    L, ns, nr = 8, 16, 2
    N = L ** 3
    even = (np.indices((L, L, L)).sum(axis=0) % 2 == 0).transpose(2, 1, 0).reshape(-1)      # i = x + L(y + Lz)
    J = np.ones((ns, 3, N), np.int8)
    # ferromagnetic ground state: every flip costs +12
    s = np.ones((ns, nr, N), np.int8)
    oracle.metropolis_checkerboard(L, s, J, seed=3, T=T, tau0=5, parity=0)
    assert np.all(s[:, :, ~even] == 1)                                 # the odd sites were not attempted
    n_att = ns * nr * N // 2
    flipped = int((s[:, :, even] == -1).sum())
    p = math.exp(-12.0 / T)
    assert abs(flipped - n_att * p) < 4.5 * math.sqrt(n_att * p * (1 - p))
    # Neel state in a ferromagnet: every bond unsatisfied, dH = -12, every attempted spin flips
    s = np.where(even, 1, -1).astype(np.int8)[None, None, :].repeat(ns, 0).repeat(nr, 1).copy()
    oracle.metropolis_checkerboard(L, s, J, seed=3, T=T, tau0=5, parity=1)
    assert np.all(s == 1)
    # one wrong neighbour each: flipping an even spin whose +x neighbour is already flipped costs +8
    s = np.ones((ns, nr, N), np.int8)
    xs = np.arange(N) % L
    s[:, :, (~even) & (xs % 4 == 1)] = -1                              # odd sites with x = 1 mod 4
    tgt = even & (xs % 4 == 0)                                         # their -x neighbours: exactly one flipped neighbour
    oracle.metropolis_checkerboard(L, s, J, seed=4, T=T, tau0=9, parity=0)
    n_att = ns * nr * int(tgt.sum())
    flipped = int((s[:, :, tgt] == -1).sum())
    p = math.exp(-8.0 / T)
    assert abs(flipped - n_att * p) < 4.5 * math.sqrt(n_att * p * (1 - p))
    # determinism and the role of the sweep index
    a = np.ones((ns, nr, N), np.int8); b = a.copy(); c = a.copy()
    oracle.metropolis_checkerboard(L, a, J, 3, T, tau0=5, n_sweeps=2)
    oracle.metropolis_checkerboard(L, b, J, 3, T, tau0=5, n_sweeps=2)
    oracle.metropolis_checkerboard(L, c, J, 3, T, tau0=6, n_sweeps=2)
    assert np.array_equal(a, b) and not np.array_equal(a, c)


@pytest.mark.parametrize("T,seed", [(2.0, 31), (3.0, 32)])
def test_checkerboard_metropolis_2x2x2_exact_boltzmann(oracle, T, seed):
    L, N, nr = 2, 8, 64
    J = random_pm1((1, 3, N), seed)
    exact = _boltzmann_2x2x2(J[0].tolist(), T)
    s = oracle.init_spins(L, 1, nr, seed)
    es = []
    for tau in range(6000):
        oracle.metropolis_checkerboard(L, s, J, seed, T, tau0=tau, n_sweeps=1)
        if tau >= 200:
            es.append(oracle.measure(L, s, np.zeros_like(s, dtype=np.uint8), J)[0] / float(N))
    per_rep = np.array(es).mean(axis=0)
    mean, err = per_rep.mean(), per_rep.std(ddof=1) / math.sqrt(nr)
    assert err < 0.01 and abs(mean - exact) < 3 * err, (mean, exact, err)


def test_checkerboard_metropolis_matches_independent_metropolis(oracle):
    """Equilibrium energy per spin at T = 2.0 on real-sized lattices against the
    typewriter-order splitmix64 Metropolis of metropolis_oracle.c (3 sigma)."""
    L, ns, nr, T = 8, 6, 2, 2.0
    N = L ** 3
    J = random_pm1((ns, 3, N), 41)
    s = random_pm1((ns, nr, N), 42)
    s_ind = s.copy()
    es = []
    for tau in range(700):
        oracle.metropolis_checkerboard(L, s, J, 7, T, tau0=tau, n_sweeps=1)
        if tau >= 200:
            es.append(oracle.measure(L, s, np.zeros_like(s, dtype=np.uint8), J)[0] / float(N))
    e_chk = np.array(es).mean(axis=0)
    e_ind = oracle.metropolis(L, s_ind, J, T, 700, seed=5)[200:].mean(axis=0)
    d = e_chk.mean() - e_ind.mean()
    err = math.sqrt(e_chk.var(ddof=1) / e_chk.size + e_ind.var(ddof=1) / e_ind.size)
    assert abs(d) < 3 * err + 2e-3, (d, err)


# ---------------------------------------------------------------- gamma daemons per spin
def test_gamma_families_are_independent_and_alpha0_is_the_single_daemon(oracle):
    L, ns, nr = 6, 3, 2
    N = L ** 3
    a = np.zeros((ns, nr, N), np.uint8); b = np.zeros_like(a); c = np.zeros_like(a)
    oracle.refresh(L, a, 11, 1.5, 4)
    oracle.refresh_alpha(L, b, 11, 1.5, 4, 0)
    oracle.refresh_alpha(L, c, 11, 1.5, 4, 3)
    np.testing.assert_array_equal(a, b)
    assert not np.array_equal(a, c)
    x, y = a.astype(np.float64).ravel() - a.mean(), c.astype(np.float64).ravel() - c.mean()
    corr = float((x * y).sum() / math.sqrt((x * x).sum() * (y * y).sum()))
    assert abs(corr) < 5 / math.sqrt(x.size)
    assert abs(4.0 * c.mean() - eq12(1.5)) < 0.05


@pytest.mark.parametrize("gamma", [2, 6])
def test_gamma_daemons_conserve_energy_and_reach_boltzmann_on_2x2x2(oracle, gamma):
    """A timestep of gamma sweeps, the alpha-th with its own daemon family: the
    total H_EA + sum_alpha H_aux,alpha is conserved between refreshes and the
    long-run energy is the exact Boltzmann average (same pin as P7)."""
    L, N, nr, T, seed = 2, 8, 64, 2.0, 58        # (sample 57 is non-ergodic on 2x2x2 for every gamma, 1 included)
    J = random_pm1((1, 3, N), seed)
    exact = _boltzmann_2x2x2(J[0].tolist(), T)
    s = oracle.init_spins(L, 1, nr, seed)
    m = np.zeros((gamma, 1, nr, N), dtype=np.uint8)
    out = driver.anneal(L, s, m, J, seed, [(T, 10, 1)] * 400)
    tot = out["E"] + out["Edem"]
    for k in range(400):                                   # constant inside every refresh interval
        blk = tot[10 * k:10 * k + 10]
        assert np.all(blk == blk[0])
    e = out["E"][200:] / float(N)
    per_rep = e.mean(axis=0)
    mean, err = per_rep.mean(), per_rep.std(ddof=1) / math.sqrt(nr)
    assert err < 0.012 and abs(mean - exact) < 3 * err, (mean, exact, err)


def test_six_walkers_conserve_energy_and_reach_boltzmann_on_2x2x2(oracle):
    """gamma = 6 walkers with the six wandering directions of Eq. (13)."""
    L, N, nr, T, seed = 2, 8, 64, 2.0, 58
    J = random_pm1((1, 3, N), seed)
    exact = _boltzmann_2x2x2(J[0].tolist(), T)
    s = oracle.init_spins(L, 1, nr, seed)
    m = np.zeros((6, 1, nr, N), dtype=np.uint8)
    out = driver.anneal(L, s, m, J, seed, [(T, 10, 1)] * 400, walkers=True)
    tot = out["E"] + out["Edem"]
    for k in range(400):
        blk = tot[10 * k:10 * k + 10]
        assert np.all(blk == blk[0])
    per_rep = (out["E"][200:] / float(N)).mean(axis=0)
    mean, err = per_rep.mean(), per_rep.std(ddof=1) / math.sqrt(nr)
    assert err < 0.012 and abs(mean - exact) < 3 * err, (mean, exact, err)
    # on a larger lattice the walkers change the trajectory (they are not daemons)
    L2 = 6
    s1 = oracle.init_spins(L2, 2, 2, 3); Jb = oracle.init_bonds(L2, 2, 3); s2 = s1.copy()
    m1 = np.zeros((6, 2, 2, L2 ** 3), np.uint8); m2 = m1.copy()
    driver.anneal(L2, s1, m1, Jb, 3, [(1.5, 4, 0)], walkers=True)
    driver.anneal(L2, s2, m2, Jb, 3, [(1.5, 4, 0)], walkers=False)
    assert not np.array_equal(s1, s2)
