"""Pins for the CPU oracle (-m "not gpu").

Each test checks oracle/ against something the paper or the mathematics fixes
and that is NOT the oracle's own formula retyped:

  P1  28-row truth table of Eq. (8)+(10)      tests/golden/truth_table.txt
  P2  exact conservation of H_EA + H_aux
  P3  the move is an involution
  P4  incremental dE == from-scratch energy   BASELINE.json north_star
  --  measure == np.roll evaluation of Eq. 1
  P6  Philox4x32-10 == cuRAND host generator  (library pin)
"""
import ctypes
from pathlib import Path

import numpy as np
import pytest

from micsa_workloads import random_levels, random_pm1

GOLDEN = Path(__file__).parent / "golden"


def _state(L, ns, nr, seed):
    N = L ** 3
    s = random_pm1((ns, nr, N), seed)
    J = random_pm1((ns, 3, N), seed + 1)
    m = random_levels((ns, nr, N), seed + 2)
    return s, m, J


def _energy_np(L, s, J):
    """Eq. (1) with np.roll: independent of the oracle's index arithmetic."""
    ns, nr, N = s.shape
    S = s.reshape(ns, nr, L, L, L).astype(np.int64)          # [.., z, y, x]
    JJ = J.reshape(ns, 3, L, L, L).astype(np.int64)
    E = np.zeros((ns, nr), dtype=np.int64)
    for d, axis in enumerate((4, 3, 2)):                      # x, y, z
        nb = np.roll(S, -1, axis=axis)                        # s[i + d]
        E -= (JJ[:, d][:, None] * S * nb).sum(axis=(2, 3, 4))
    return E.reshape(-1)


# ---------------------------------------------------------------- P6 Philox
def _curand():
    for name in ("libcurand.so.10", "libcurand.so",
                 "/usr/local/cuda/lib64/libcurand.so.10"):
        try:
            return ctypes.CDLL(name)
        except OSError:
            continue
    return None


@pytest.mark.parametrize("seed,offset", [(0, 0), (0x0123456789ABCDEF, 0),
                                         (1, 4 * 12345), (1, 4 * 65536 * 77 + 4 * 65530),
                                         (2**63 + 17, 4 * 65536 * (2**32 + 5) + 4 * 9)])
def test_philox_matches_curand_host(oracle, seed, offset):
    cr = _curand()
    if cr is None:
        pytest.skip("libcurand not loadable")
    gen = ctypes.c_void_p()
    CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
    assert cr.curandCreateGeneratorHost(ctypes.byref(gen), CURAND_RNG_PSEUDO_PHILOX4_32_10) == 0
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    assert cr.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
    n_sub = 64
    out = (ctypes.c_uint32 * (4 * n_sub))()
    assert cr.curandGenerate(gen, out, ctypes.c_size_t(4 * n_sub)) == 0
    cr.curandDestroyGenerator(gen)
    got = np.frombuffer(out, dtype=np.uint32).reshape(n_sub, 4)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    # cuRAND host ordering (found empirically, CUDA 12.9): the stream interleaves
    # 65536 subsequences; quadruple number q = offset/4 + k is
    # Philox(counter = (q / 65536 as 64 bit, q % 65536 as 64 bit), key = seed).
    # The host API therefore exercises c0, c1, the low 16 bits of c2 and both
    # key words; c3 and the rest of c2 are covered by the all-words test below
    # and by the device-API pin test_philox_matches_curand_device_api in
    # tests/test_gpu_parity.py (curand_init's subsequence reaches c2 and c3).
    for k in range(n_sub):
        q = offset // 4 + k
        pos, sub = q // 65536, q % 65536
        ctr = (pos & 0xFFFFFFFF, pos >> 32, sub, 0)
        np.testing.assert_array_equal(oracle.philox4x32_10(ctr, key), got[k])


def test_philox_counter_words_all_matter(oracle):
    base = oracle.philox4x32_10((1, 2, 3, 4), (5, 6))
    for w in range(4):
        c = [1, 2, 3, 4]
        c[w] += 1
        assert not np.array_equal(oracle.philox4x32_10(c, (5, 6)), base)
    assert not np.array_equal(oracle.philox4x32_10((1, 2, 3, 4), (5, 7)), base)
    assert not np.array_equal(oracle.philox4x32_10((1, 2, 3, 4), (6, 6)), base)


# ---------------------------------------------------------------- P1 truth table
def _single_site_case(oracle, U, m0, spin, pattern_seed):
    """L=4 lattice, site (1,1,1) (odd parity) with exactly U unsatisfied bonds."""
    L, N = 4, 64
    rng = np.random.default_rng(pattern_seed)
    s = random_pm1((1, 1, N), pattern_seed)
    J = random_pm1((1, 3, N), pattern_seed + 7)
    m = random_levels((1, 1, N), pattern_seed + 9)
    idx = lambda x, y, z: (x % L) + L * ((y % L) + L * (z % L))
    x = y = z = 1
    i = idx(x, y, z)
    s[0, 0, i] = spin
    m[0, 0, i] = m0
    # (neighbour index, bond array d, bond owner site)
    nbrs = [(idx(x + 1, y, z), 0, i), (idx(x - 1, y, z), 0, idx(x - 1, y, z)),
            (idx(x, y + 1, z), 1, i), (idx(x, y - 1, z), 1, idx(x, y - 1, z)),
            (idx(x, y, z + 1), 2, i), (idx(x, y, z - 1), 2, idx(x, y, z - 1))]
    unsat = set(rng.choice(6, size=U, replace=False).tolist())
    for k, (j, d, owner) in enumerate(nbrs):
        # bond satisfied <=> J s_i s_j = +1
        want = -1 if k in unsat else +1
        J[0, d, owner] = want * spin * s[0, 0, j]
    return L, s, m, J, i


def test_truth_table(oracle):
    table = np.loadtxt(GOLDEN / "truth_table.txt", dtype=int)
    assert table.shape == (28, 4) and table[:, 2].sum() == 16
    for U, m0, acc, m_new in table:
        for spin in (-1, +1):
            for pat in range(4):
                L, s, m, J, i = _single_site_case(oracle, U, m0, spin, 100 * U + 10 * m0 + pat)
                s0, m0_all = s.copy(), m.copy()
                oracle.half_sweep(L, s, m, J, 1)          # (1,1,1) is an odd site
                assert s[0, 0, i] == (-spin if acc else spin), (U, m0, spin)
                assert m[0, 0, i] == m_new, (U, m0, spin)
                # even sites untouched by the odd half-sweep
                xs = np.arange(64)
                par = ((xs % 4) + (xs // 4) % 4 + xs // 16) % 2
                np.testing.assert_array_equal(s[0, 0, par == 0], s0[0, 0, par == 0])
                np.testing.assert_array_equal(m[0, 0, par == 0], m0_all[0, 0, par == 0])


# ---------------------------------------------------------------- measure
@pytest.mark.parametrize("L", [2, 4, 6])
def test_measure_matches_numpy_roll(oracle, L):
    s, m, J = _state(L, 3, 2, 11 + L)
    E, Ed, Q = oracle.measure(L, s, m, J)
    np.testing.assert_array_equal(E, _energy_np(L, s, J))
    np.testing.assert_array_equal(Ed, 4 * m.astype(np.int64).sum(axis=2).reshape(-1))
    np.testing.assert_array_equal(
        Q, (s[:, 0].astype(np.int64) * s[:, 1]).sum(axis=1))


def test_measure_ground_states(oracle):
    """Ferromagnet (all J=+1, all s=+1): E = -3N; flipping one spin costs 12."""
    L, N = 4, 64
    s = np.ones((1, 2, N), dtype=np.int8)
    J = np.ones((1, 3, N), dtype=np.int8)
    m = np.zeros((1, 2, N), dtype=np.uint8)
    s[0, 1, 5] = -1
    E, Ed, Q = oracle.measure(L, s, m, J)
    assert E.tolist() == [-3 * N, -3 * N + 12] and Ed.tolist() == [0, 0]
    assert Q.tolist() == [N - 2]


def test_q_pair_order(oracle):
    L, N = 2, 8
    s = random_pm1((2, 3, N), 5)
    m = np.zeros((2, 3, N), dtype=np.uint8)
    J = random_pm1((2, 3, N), 6)
    _, _, Q = oracle.measure(L, s, m, J)
    want = [int((s[k, a].astype(int) * s[k, b]).sum())
            for k in range(2) for (a, b) in ((0, 1), (0, 2), (1, 2))]
    assert Q.tolist() == want


# ---------------------------------------------------------------- P2, P3, P4
@pytest.mark.parametrize("L", [2, 4, 6, 8])
def test_conservation_and_incremental_energy(oracle, L):
    s, m, J = _state(L, 2, 2, 40 + L)
    E0, Ed0, _ = oracle.measure(L, s, m, J)
    tot = E0 + Ed0
    for t in range(12):
        for p in (0, 1):
            Eb, _, _ = oracle.measure(L, s, m, J)
            acc, dE = oracle.half_sweep(L, s, m, J, p)
            E, Ed, _ = oracle.measure(L, s, m, J)
            np.testing.assert_array_equal(E + Ed, tot)          # P2
            np.testing.assert_array_equal(E - Eb, dE)           # P4
            np.testing.assert_array_equal(E, _energy_np(L, s, J))
            assert m.max() <= 3
            if t == 0 and L >= 4:
                assert acc.min() > 0


@pytest.mark.parametrize("L", [2, 4, 6])
def test_involution_and_reversibility(oracle, L):
    s, m, J = _state(L, 2, 2, 70 + L)
    s0, m0 = s.copy(), m.copy()
    for p in (0, 1):
        oracle.half_sweep(L, s, m, J, p)
        assert not np.array_equal(s, s0)
        oracle.half_sweep(L, s, m, J, p)
        np.testing.assert_array_equal(s, s0)
        np.testing.assert_array_equal(m, m0)
    n = 7
    oracle.sweep(L, s, m, J, n)
    assert not np.array_equal(s, s0)
    for _ in range(n):                    # undo: odd first, then even
        oracle.half_sweep(L, s, m, J, 1)
        oracle.half_sweep(L, s, m, J, 0)
    np.testing.assert_array_equal(s, s0)
    np.testing.assert_array_equal(m, m0)


def test_half_sweep_touches_only_its_parity_and_ignores_order(oracle):
    """Sites of one parity do not interact: updating the lattice
    reflected in x (a different visiting order) gives the reflected result."""
    L = 4
    s, m, J = _state(L, 1, 1, 91)
    S = s.reshape(L, L, L); M = m.reshape(L, L, L); JJ = J.reshape(3, L, L, L)
    # reflection x -> -x mod L keeps parity; bond (x -> x+1) becomes the x-bond
    # owned by the reflected neighbour
    xs = (-np.arange(L)) % L
    Sr = np.ascontiguousarray(S[:, :, xs]).reshape(1, 1, -1)
    Mr = np.ascontiguousarray(M[:, :, xs]).reshape(1, 1, -1)
    Jr = np.empty_like(JJ)
    Jr[0] = np.roll(JJ[0], 1, axis=2)[:, :, xs]      # Jx'(x') = Jx(x-1) at x = -x'
    Jr[1] = JJ[1][:, :, xs]
    Jr[2] = JJ[2][:, :, xs]
    Jr = np.ascontiguousarray(Jr).reshape(1, 3, -1)
    oracle.sweep(L, s, m, J, 3)
    oracle.sweep(L, Sr, Mr, Jr, 3)
    np.testing.assert_array_equal(Sr.reshape(L, L, L), s.reshape(L, L, L)[:, :, xs])
    np.testing.assert_array_equal(Mr.reshape(L, L, L), m.reshape(L, L, L)[:, :, xs])


def test_sample_replica_indexing(oracle):
    """Replicas of a sample share its couplings; systems are independent."""
    L = 4
    s, m, J = _state(L, 3, 2, 123)
    s_ref, m_ref = s.copy(), m.copy()
    oracle.sweep(L, s, m, J, 5)
    for k in range(3):
        for r in range(2):
            s1 = np.ascontiguousarray(s_ref[k:k + 1, r:r + 1])
            m1 = np.ascontiguousarray(m_ref[k:k + 1, r:r + 1])
            oracle.sweep(L, s1, m1, np.ascontiguousarray(J[k:k + 1]), 5)
            np.testing.assert_array_equal(s1[0, 0], s[k, r])
            np.testing.assert_array_equal(m1[0, 0], m[k, r])


def test_paper_table3_consistency():
    """BASELINE.md's derived figures follow from Table 3."""
    t = dict((k, int(v)) for k, v in
             (l.split() for l in (GOLDEN / "paper_table3.txt").read_text().splitlines()
              if not l.startswith("#")))
    metro = t["metropolis_rng"] + t["metropolis_update"]
    mic = t["micsa_update"] + t["micsa_walk"]
    assert abs(metro / mic - 1.9) < 0.05                   # caption: "1.9 times"
    assert abs(t["micsa_walk"] / mic - 0.44) < 0.01
    assert abs(t["metropolis_rng"] / metro - 0.72) < 0.01
    attempts = 160 ** 3 * 128
    assert abs(mic * 1e3 / attempts - 0.4) < 0.02          # "~0.4 ps"


# ---------------------------------------------------------------- C4 (Eq. 16)
@pytest.mark.parametrize("L,ns,nr", [(4, 2, 2), (6, 1, 3), (8, 2, 2)])
def test_c4_against_numpy_roll_and_identities(oracle, L, ns, nr):
    N = L ** 3
    s = random_pm1((ns, nr, N), 91)
    S = oracle.c4(L, s)
    assert S.shape == (ns * nr * (nr - 1) // 2, 3, L // 2 + 1)
    k = 0
    for sample in range(ns):
        for a in range(nr):
            for b in range(a + 1, nr):
                q = (s[sample, a].astype(np.int64) * s[sample, b]).reshape(L, L, L)      # [z, y, x]
                for d, ax in enumerate((2, 1, 0)):                                      # x is the last numpy axis
                    for r in range(L // 2 + 1):
                        assert S[k, d, r] == int((q * np.roll(q, -r, axis=ax)).sum())
                    # sum over all displacements along the axis = sum of squared line sums
                    full = sum(int((q * np.roll(q, -r, axis=ax)).sum()) for r in range(L))
                    assert full == int((q.sum(axis=ax) ** 2).sum())
                    # S(r) = S(L - r): the half range holds everything
                    assert full == int(S[k, d, 0] + 2 * S[k, d, 1:L // 2].sum() + S[k, d, L // 2])
                assert np.all(S[k, :, 0] == N)
                k += 1
    same = np.repeat(random_pm1((1, 1, N), 92), 2, axis=1)                              # identical replicas
    assert np.all(oracle.c4(L, same) == N)
    stag = np.where(np.indices((L, L, L)).sum(axis=0) % 2 == 0, 1, -1).astype(np.int8).reshape(1, 1, N)
    pair = np.concatenate([stag, np.ones((1, 1, N), np.int8)], axis=1)                  # q = staggered field
    want = np.array([N * (-1) ** r for r in range(L // 2 + 1)])
    assert np.all(oracle.c4(L, pair)[0] == want[None, :])


# ---------------------------------------------------------------- I_n, xi_12, xi_23 / xi_12 (Eq. 17-18)
def test_xi_closed_forms(oracle):
    """Eq. (17)-(18) under reading R22 (trapezoid on the lattice, cut where C4 first drops to the floor, no tail).
    For C4(r) = exp(-r / xi) the continuum integrals are I_n = n! xi^(n+1), so xi_12 = 2 xi and xi_23 / xi_12 = 3/2;
    the trapezoid on integer r differs at relative order 1 / xi^2.  The trapezoid itself has a closed form for a
    triangle C4(r) = 1 - r / R."""
    for x in (6.0, 10.0, 25.0):
        r = np.arange(40 * int(x))
        I1, I2, I3, xi12, ratio = oracle.xi(np.exp(-r / x))
        tol = 0.5 / x ** 2
        assert abs(I1 / x ** 2 - 1.0) < tol and abs(I2 / (2 * x ** 3) - 1.0) < tol and abs(I3 / (6 * x ** 4) - 1.0) < tol
        assert abs(xi12 / (2 * x) - 1.0) < tol and abs(ratio / 1.5 - 1.0) < tol
    R = 12
    tri = 1.0 - np.arange(R + 1) / R
    I1 = oracle.xi(tri, c_min=-1.0)[0]                       # trapezoid of r (1 - r/R) on [0, R]: sum_{r=1}^{R-1} r (1 - r/R)
    assert abs(I1 - sum(k * (1 - k / R) for k in range(1, R))) < 1e-12
    # the cut-off: values after the first one at or below the floor do not enter, wherever they are
    c = np.exp(-np.arange(30) / 3.0)
    noisy = c.copy(); noisy[14] = -1e-3; noisy[15:] = 5.0
    np.testing.assert_allclose(oracle.xi(noisy), oracle.xi(c[:14]), rtol=1e-15)
    np.testing.assert_allclose(oracle.xi(c, c_min=c[9]), oracle.xi(c[:9]), rtol=1e-15)
    with pytest.raises(ValueError):
        oracle.xi(np.array([1.0, 0.0, 0.5]))


def test_c4_normalisation_over_all_replica_pairs(oracle):
    """Eq. (16) sums over every pair a != b with N~ = N N_R (N_R - 1) / 2: with three replicas of
    which two are identical and one independent, C4(0) = 1 and the pair of identical replicas contributes exactly 1 at
    every r, so C4(r) = (1 + 2 c(r)) / 3 with c the two-replica value of the mixed pairs."""
    L, N = 8, 512
    a = random_pm1((1, 1, N), 101); b = random_pm1((1, 1, N), 102)
    s3 = np.ascontiguousarray(np.concatenate([a, a, b], axis=1))
    S3 = oracle.c4(L, s3)
    assert S3.shape == (3, 3, L // 2 + 1)                    # pairs (0,1), (0,2), (1,2)
    assert np.all(S3[0] == N) and np.array_equal(S3[1], S3[2])
    c2 = oracle.c4_normalised(L, oracle.c4(L, np.ascontiguousarray(np.concatenate([a, b], axis=1))))
    c3 = oracle.c4_normalised(L, S3)
    np.testing.assert_allclose(c3, (1.0 + 2.0 * c2) / 3.0, rtol=1e-14)
    assert c3[0] == 1.0


def test_xi_grows_in_a_quench(oracle):
    """PAPER.md:283, Fig. 2: below T_c the coherence length xi_12(t) grows with time.  L = 12, T = 0.7, 8 samples x 2
    replicas of the oracle's MicSA dynamics: xi_12 after 64 sweeps exceeds xi_12 after 4, and C4(0) = 1."""
    from oracle import driver
    L, ns, nr, seed = 12, 8, 2, 5
    s = oracle.init_spins(L, ns, nr, seed); J = oracle.init_bonds(L, ns, seed)
    m = np.zeros_like(s, dtype=np.uint8)
    out = []
    done = 0
    for t_end in (4, 64):
        driver.anneal(L, s, m, J, seed, [(0.7, 4, 0)] * ((t_end - done) // 4), step0=done // 4)
        done = t_end
        S = oracle.c4(L, s)                                  # one pair per sample
        c4 = np.mean([oracle.c4_normalised(L, S[k:k + 1]) for k in range(ns)], axis=0)
        assert c4[0] == 1.0
        out.append(oracle.xi(c4, c_min=0.01)[3])
    assert out[1] > 1.15 * out[0] > 0.0, out
