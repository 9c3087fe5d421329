"""Pins of the continuous-daemon / Gaussian-coupling oracle (oracle/gauss_oracle.c).
All -m "not gpu": the oracle is checked against what the paper and the mathematics fix, not against itself.

P15  refresh: Kolmogorov-Smirnov of n against Eq. (9), Prob(n < R) = 1 - exp(-R/T), mean T,
     variance T^2, n = -T log(u) with the uniform of the documented Philox counter
P16  the move conserves H_EA + sum n: to rounding with Gaussian J, EXACTLY with J = +-1 and integer n;
     it is its own inverse; dH is Eq. (1)'s energy difference (np.roll evaluation)
P17  with J = +-1, n = 4m and daemons that never exceed the cap, it is the capped integer move of micsa_oracle.c
P18  2x2x2 lattice, Gaussian J: long-run <e> against the exact Boltzmann average over all 2^8 states, T = 2, 3
P19  equilibrium energy at L = 4 against an independent Metropolis written here in numpy
P20  wandering: exchange twice = identity, period L
"""
import itertools

import numpy as np

from micsa_workloads import gaussian_couplings, random_pm1


def _energy_roll(L, s, J):
    """Eq. (1) per system with np.roll, independent of the oracle's loops."""
    ns, nr, N = s.shape
    S = s.reshape(ns, nr, L, L, L).astype(np.float64)       # [z][y][x]
    JJ = J.reshape(ns, 3, L, L, L)
    E = np.zeros((ns, nr))
    for d, ax in ((0, 4), (1, 3), (2, 2)):
        E -= (JJ[:, d][:, None] * S * np.roll(S, -1, axis=ax)).sum(axis=(2, 3, 4))
    return E.reshape(-1)


def test_refresh_is_exponential_eq9(oracle):
    L, ns, nr, seed = 16, 4, 2, 77
    for T, step in [(2.0, 0), (0.2, 5)]:
        n = np.zeros((ns, nr, L ** 3))
        oracle.gauss_refresh(L, n, seed, T, step, sample_offset=3)
        x = np.sort(n.reshape(-1))
        cdf = 1.0 - np.exp(-x / T)                             # Eq. (9)
        m = x.size
        ks = max(np.max(np.arange(1, m + 1) / m - cdf), np.max(cdf - np.arange(m) / m))
        assert ks < 1.63 / np.sqrt(m)                          # 1 % level
        assert abs(x.mean() / T - 1.0) < 5.0 / np.sqrt(m)
        assert abs(x.var() / T ** 2 - 1.0) < 5.0 * np.sqrt(8.0 / m)
        assert x.min() > 0.0
        # the documented map: n = -T log(u), u = (word + 1/2) 2^-32 of counter (i, sample, tag|replica, step)
        for (sa, r, i) in [(0, 0, 0), (3, 1, 4095), (2, 0, 1234)]:
            u = oracle.gauss_uniform(i, 3 + sa, r, step, seed)
            assert 0.0 < u < 1.0
            assert n[sa, r, i] == -T * np.log(u)
    # same counters, same numbers; another step, other numbers
    a = np.zeros((1, 1, 64)); b = np.zeros((1, 1, 64)); c = np.zeros((1, 1, 64))
    oracle.gauss_refresh(4, a, 1, 1.0, 7); oracle.gauss_refresh(4, b, 1, 1.0, 7); oracle.gauss_refresh(4, c, 1, 1.0, 8)
    assert np.array_equal(a, b) and not np.array_equal(a, c)


def test_conservation_and_energy_difference(oracle):
    L, ns, nr = 6, 3, 2
    N = L ** 3
    s = random_pm1((ns, nr, N), 1)
    J = gaussian_couplings((ns, 3, N), 2)
    n = np.zeros((ns, nr, N))
    oracle.gauss_refresh(L, n, 5, 1.5, 0)
    E0, Ed0, _ = oracle.gauss_measure(L, s, n, J)
    np.testing.assert_allclose(E0, _energy_roll(L, s, J), rtol=1e-12)
    np.testing.assert_allclose(Ed0, n.sum(axis=2).reshape(-1), rtol=1e-12)
    for t in range(5):
        for p in (0, 1):
            s_before = s.copy()
            oracle.gauss_half_sweep(L, s, n, J, p)
            E, Ed, _ = oracle.gauss_measure(L, s, n, J)
            np.testing.assert_allclose(E + Ed, E0 + Ed0, rtol=0, atol=1e-9)
            np.testing.assert_allclose(E, _energy_roll(L, s, J), rtol=1e-12)
            assert n.min() >= 0.0
            assert not np.array_equal(s, s_before)
    assert np.all(E < E0)                                      # a quench relaxes


def test_exact_with_integer_energies_and_involution(oracle):
    """J = +-1 and integer n: every quantity is an integer in float64, so conservation and the involution are EXACT."""
    L, ns, nr = 4, 2, 2
    N = L ** 3
    s = random_pm1((ns, nr, N), 3)
    J = random_pm1((ns, 3, N), 4).astype(np.float64)
    n = 4.0 * np.random.default_rng(5).integers(0, 6, size=(ns, nr, N)).astype(np.float64)
    E0, Ed0, _ = oracle.gauss_measure(L, s, n, J)
    s0, n0 = s.copy(), n.copy()
    for p in (0, 1):
        oracle.gauss_half_sweep(L, s, n, J, p)
        E, Ed, _ = oracle.gauss_measure(L, s, n, J)
        assert np.array_equal(E + Ed, E0 + Ed0)
        oracle.gauss_half_sweep(L, s, n, J, p)                 # the move undoes itself
        assert np.array_equal(s, s0) and np.array_equal(n, n0)
    oracle.gauss_sweep(L, s, n, J, 7)
    for _ in range(7):
        oracle.gauss_half_sweep(L, s, n, J, 1); oracle.gauss_half_sweep(L, s, n, J, 0)
    assert np.array_equal(s, s0) and np.array_equal(n, n0)


def test_reduces_to_the_capped_integer_move(oracle):
    """the cap n <= 12 is the only difference between Sec. 2.3 and Sec. 2.5.  With J = +-1 the
    daemons stay multiples of 4; sites whose n - dH stays <= 12 move identically, and a site where the integer oracle
    rejects because of the cap is exactly a site where the uncapped move produced n > 12."""
    L, ns, nr = 6, 2, 2
    N = L ** 3
    s = random_pm1((ns, nr, N), 13); Ji = random_pm1((ns, 3, N), 14)
    m = np.random.default_rng(15).integers(0, 4, size=(ns, nr, N)).astype(np.uint8)
    for p in (0, 1):
        si, mi = s.copy(), m.copy()
        oracle.half_sweep(L, si, mi, Ji, p)
        sc, nc = s.copy(), 4.0 * m.astype(np.float64)
        oracle.gauss_half_sweep(L, sc, nc, Ji.astype(np.float64), p)
        over = nc > 12.0
        assert over.any()
        same = ~over
        assert np.array_equal(sc[same], si[same]) and np.array_equal(nc[same], 4.0 * mi[same])
        assert np.array_equal(si[over], s[over]) and np.array_equal(mi[over], m[over])      # capped: rejected
        s, m = si, mi


def _exact_boltzmann_2x2x2(J, T):
    """<e> over all 2^8 states of the 24-bond 2x2x2 periodic lattice (R10)."""
    L, N = 2, 8
    es, ws = [], []
    for bits in itertools.product((-1, 1), repeat=N):
        s = np.array(bits, dtype=np.int8).reshape(1, 1, N)
        e = _energy_roll(L, s, J[None])[0]
        es.append(e); ws.append(np.exp(-e / T))
    es, ws = np.array(es), np.array(ws)
    return float((es * ws).sum() / ws.sum() / N)


def test_boltzmann_average_2x2x2_gaussian(oracle):
    """Stationarity of refresh + sweeps: the canonical average of the spin energy."""
    L, N = 2, 8
    ns, nr = 16, 4                                            # independent chains of the same sample
    Js = gaussian_couplings((3, N), 21)
    J = np.ascontiguousarray(np.broadcast_to(Js, (ns, 3, N)))
    for T, seed in [(2.0, 31), (3.0, 32)]:
        exact = _exact_boltzmann_2x2x2(Js, T)
        s = random_pm1((ns, nr, N), seed)
        n = np.zeros((ns, nr, N))
        acc = []
        for k in range(2500):
            oracle.gauss_refresh(L, n, seed, T, k)
            oracle.gauss_sweep(L, s, n, J, 3)
            if k >= 100:
                acc.append(oracle.gauss_measure(L, s, n, J)[0] / N)
        a = np.array(acc)                                     # [time, chain]
        per_chain = a.mean(axis=0)
        err = per_chain.std(ddof=1) / np.sqrt(per_chain.size)
        assert abs(per_chain.mean() - exact) < 3.5 * err + 1e-3, (T, per_chain.mean(), exact, err)


def _metropolis_numpy(L, s, J, T, n_sweeps, rng):
    """Independent single-spin-flip Metropolis (typewriter order) for one system; returns e per sweep."""
    N = L ** 3
    S = s.reshape(L, L, L).astype(np.float64).copy()          # [z][y][x]
    JJ = J.reshape(3, L, L, L)
    out = []
    for _ in range(n_sweeps):
        for z in range(L):
            for y in range(L):
                for x in range(L):
                    h = (JJ[0, z, y, x] * S[z, y, (x + 1) % L] + JJ[0, z, y, x - 1] * S[z, y, x - 1]
                         + JJ[1, z, y, x] * S[z, (y + 1) % L, x] + JJ[1, z, y - 1, x] * S[z, y - 1, x]
                         + JJ[2, z, y, x] * S[(z + 1) % L, y, x] + JJ[2, z - 1, y, x] * S[z - 1, y, x])
                    dH = 2.0 * S[z, y, x] * h
                    if dH <= 0.0 or rng.random() < np.exp(-dH / T):
                        S[z, y, x] = -S[z, y, x]
        e = 0.0
        for d, ax in ((0, 2), (1, 1), (2, 0)):
            e -= (JJ[d] * S * np.roll(S, -1, axis=ax)).sum()
        out.append(e / N)
    return np.array(out)


def test_equilibrium_energy_against_independent_metropolis(oracle):
    L, N, T = 4, 64, 2.0
    Js = gaussian_couplings((3, N), 41)
    rng = np.random.default_rng(42)
    met = np.array([_metropolis_numpy(L, random_pm1((N,), 50 + c), Js, T, 260, rng)[60:].mean() for c in range(6)])
    ns, nr = 12, 4
    J = np.ascontiguousarray(np.broadcast_to(Js, (ns, 3, N)))
    s = random_pm1((ns, nr, N), 43)
    n = np.zeros((ns, nr, N))
    acc = []
    for k in range(400):
        oracle.gauss_refresh(L, n, 44, T, k)
        oracle.gauss_sweep(L, s, n, J, 2)
        if k >= 50:
            acc.append(oracle.gauss_measure(L, s, n, J)[0] / N)
    mic = np.array(acc).mean(axis=0)
    err = np.sqrt(mic.var(ddof=1) / mic.size + met.var(ddof=1) / met.size)
    assert abs(mic.mean() - met.mean()) < 3.5 * err + 2e-3, (mic.mean(), met.mean(), err)


def test_wandering_period_and_involution(oracle):
    L, ns, nr = 6, 2, 2
    lab = np.random.default_rng(61).random((ns, nr, L ** 3))
    n = lab.copy()
    oracle.gauss_wander(L, n, 0, +1, 0)
    assert not np.array_equal(n, lab) and np.array_equal(np.sort(n, axis=2), np.sort(lab, axis=2))
    oracle.gauss_wander(L, n, 0, +1, 0)
    assert np.array_equal(n, lab)
    for t in range(L):                                        # L half-cycles bring every walker home
        oracle.gauss_wander(L, n, 0, +1, t & 1)
    assert np.array_equal(n, lab)
    # conservation with walkers: the exchange only permutes the n
    s = random_pm1((ns, nr, L ** 3), 62); J = gaussian_couplings((ns, 3, L ** 3), 63)
    E0, Ed0, _ = oracle.gauss_measure(L, s, n, J)
    oracle.gauss_sweep(L, s, n, J, 5, walkers=True, t0=3)
    E, Ed, _ = oracle.gauss_measure(L, s, n, J)
    np.testing.assert_allclose(E + Ed, E0 + Ed0, atol=1e-9)
