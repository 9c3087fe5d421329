"""Parity of the continuous-daemon CUDA path (micsa_gauss_*) with oracle/gauss_oracle.c (-m gpu).

Tolerance reading (R18-R21): the move's arithmetic (local field, dH, n - dH, the accept decision) is the same
sequence of separately rounded float64 operations on both sides, so from identical inputs spins AND daemon energies
are bit-identical; only the refresh goes through log(), where the CUDA and the C library may differ in the last place:
refreshed n are compared to 1e-14 relative, and what follows a device refresh to 1e-12 (spins still exactly: a flipped
decision would need |n - dH| below 1e-15).  E and E_daemon are float64 sums in another order: 1e-12 of sum |terms|.
"""
import numpy as np
import pytest

from micsa_workloads import gaussian_couplings, random_pm1

pytestmark = pytest.mark.gpu

SHAPES = [(2, 1, 2), (4, 3, 2), (6, 5, 3), (8, 2, 1), (10, 4, 2), (16, 3, 2)]


def _assert_exact(g, s, n):
    gs, gn, _ = g.get_state(couplings=False)
    np.testing.assert_array_equal(gs, s)
    np.testing.assert_array_equal(gn, n)


@pytest.mark.parametrize("L,ns,nr", SHAPES)
def test_gauss_init_and_roundtrip(micsa, oracle, L, ns, nr):
    N = L ** 3
    for seed, off in [(1, 0), (0xDEADBEEF12345678, 37)]:
        with micsa.GaussMicSA(L, ns, nr, seed, sample_offset=off) as g:
            s, n, J = g.get_state()
            np.testing.assert_array_equal(s, oracle.init_spins(L, ns, nr, seed, off))      # the same Philox start
            assert not n.any() and not J.any()
            J2 = gaussian_couplings((ns, 3, N), 3); s2 = random_pm1((ns, nr, N), 4)
            n2 = np.random.default_rng(5).exponential(1.3, size=(ns, nr, N))
            g.set_couplings(J2); g.set_state(s2, n2)
            gs, gn, gJ = g.get_state()
            np.testing.assert_array_equal(gs, s2); np.testing.assert_array_equal(gn, n2); np.testing.assert_array_equal(gJ, J2)


@pytest.mark.parametrize("L,ns,nr", SHAPES)
def test_gauss_sweeps_bit_exact(micsa, oracle, L, ns, nr):
    N = L ** 3
    s = random_pm1((ns, nr, N), 11); J = gaussian_couplings((ns, 3, N), 12)
    n = np.random.default_rng(13).exponential(0.8, size=(ns, nr, N))
    with micsa.GaussMicSA(L, ns, nr, 1) as g:
        g.set_couplings(J); g.set_state(s, n)
        for t in range(4):
            for p in (0, 1):
                g.half_sweep(p); oracle.gauss_half_sweep(L, s, n, J, p)
                _assert_exact(g, s, n)
        g.sweep(6); oracle.gauss_sweep(L, s, n, J, 6)
        _assert_exact(g, s, n)
        assert g.counters()["attempts"] == 10 * N * ns * nr
        E, Ed, Q = g.measure()
        oE, oEd, oQ = oracle.gauss_measure(L, s, n, J)
        scale = np.abs(J).sum(axis=(1, 2)).repeat(nr)
        np.testing.assert_allclose(E, oE, rtol=0, atol=1e-12 * scale.max())
        np.testing.assert_allclose(Ed, oEd, rtol=1e-12)
        np.testing.assert_array_equal(Q, oQ)


@pytest.mark.parametrize("L,ns,nr", SHAPES)
def test_gauss_refresh_and_walkers(micsa, oracle, L, ns, nr):
    """Appendix C's fixed-temperature move: refresh from Eq. (9), then sweeps alternating with the forward-X wandering."""
    N = L ** 3
    seed, off = 21, 5
    J = gaussian_couplings((ns, 3, N), 22)
    s = oracle.init_spins(L, ns, nr, seed, off)
    n = np.zeros((ns, nr, N))
    with micsa.GaussMicSA(L, ns, nr, seed, sample_offset=off) as g:
        g.set_couplings(J)
        g.set_walkers(1, 0)
        t = 0
        for k, T in enumerate((2.0, 1.1, 0.2)):
            g.refresh(T, k); oracle.gauss_refresh(L, n, seed, T, k, off)
            gn = g.get_state(spins=False, couplings=False)[1]
            np.testing.assert_allclose(gn, n, rtol=1e-14, atol=0)
            assert gn.min() > 0.0
            g.sweep(5); oracle.gauss_sweep(L, s, n, J, 5, walkers=True, t0=t); t += 5
            gs, gn, _ = g.get_state(couplings=False)
            np.testing.assert_array_equal(gs, s)
            np.testing.assert_allclose(gn, n, rtol=1e-12, atol=1e-13)
            g.set_state(None, n)                               # re-synchronise the last place for the exact checks below
        assert g.counters()["rns_drawn"] == 3 * N * ns * nr
        # single half-cycles, every axis and direction, exactly
        g.set_state(s, n)
        for axis in (0, 1, 2):
            for sign in (1, -1):
                for parity in (0, 1):
                    g.wander(axis, sign, parity); oracle.gauss_wander(L, n, axis, sign, parity)
                    _assert_exact(g, s, n)
        # an odd starting time, walkers off again
        g.set_walkers(1, 7); g.sweep(2); oracle.gauss_sweep(L, s, n, J, 2, walkers=True, t0=7)
        _assert_exact(g, s, n)
        g.set_walkers(0, 0); g.sweep(2); oracle.gauss_sweep(L, s, n, J, 2)
        _assert_exact(g, s, n)


def test_gauss_conservation_and_reversal_on_gpu(micsa):
    """P16 on the device at L = 32: H_EA + sum n conserved to rounding, 20 sweeps forward + 20 reversed restore the spins
    (and the daemons to rounding)."""
    L, ns, nr = 32, 4, 2
    N = L ** 3
    with micsa.GaussMicSA(L, ns, nr, 3) as g:
        g.set_couplings(gaussian_couplings((ns, 3, N), 31))
        g.refresh(0.7, 0)
        s0, n0, _ = g.get_state(couplings=False)
        E0, Ed0, _ = g.measure()
        g.sweep(20)
        E1, Ed1, _ = g.measure()
        np.testing.assert_allclose(E1 + Ed1, E0 + Ed0, rtol=1e-11)
        assert np.all(E1 < E0)
        for _ in range(20):
            g.half_sweep(1); g.half_sweep(0)
        s1, n1, _ = g.get_state(couplings=False)
        np.testing.assert_array_equal(s1, s0)
        np.testing.assert_allclose(n1, n0, rtol=0, atol=1e-12)


def test_gauss_appendix_c_shape(micsa, oracle):
    """The shape of the paper's Appendix C run: L = 10, Gaussian couplings, N_R = 2 replicas of
    N_beta = 40 clones at temperatures uniform in [0.2, 2] -- here 40 'samples' sharing one coupling realisation, each
    refreshed at its own temperature -- one walker per spin refreshed at every EMCS, 10 x (sweep + forward-X
    wandering).  Three EMCS against the oracle; no parallel tempering / Houdayer step (out of scope)."""
    L, n_beta, nr = 10, 40, 2
    N = L ** 3
    Js = gaussian_couplings((3, N), 41)
    J = np.ascontiguousarray(np.broadcast_to(Js, (n_beta, 3, N)))
    temps = np.linspace(0.2, 2.0, n_beta)
    ctxs = [micsa.GaussMicSA(L, 1, nr, 77, sample_offset=b) for b in range(n_beta)]
    try:
        states = []
        for b, g in enumerate(ctxs):
            g.set_couplings(J[b:b + 1]); g.set_walkers(1, 0)
            states.append((oracle.init_spins(L, 1, nr, 77, b), np.zeros((1, nr, N))))
        for emcs in range(3):
            for b, g in enumerate(ctxs):
                s, n = states[b]
                g.refresh(temps[b], emcs); oracle.gauss_refresh(L, n, 77, temps[b], emcs, b)
                g.sweep(10); oracle.gauss_sweep(L, s, n, J[b:b + 1], 10, walkers=True, t0=10 * emcs)
                gs, gn, _ = g.get_state(couplings=False)
                np.testing.assert_array_equal(gs, s)
                np.testing.assert_allclose(gn, n, rtol=1e-12, atol=1e-13)
                g.set_state(None, n)
        E, _, Q = ctxs[0].measure()
        oE, _, oQ = oracle.gauss_measure(L, states[0][0], states[0][1], J[0:1])
        np.testing.assert_allclose(E, oE, rtol=1e-12)
        np.testing.assert_array_equal(Q, oQ)
    finally:
        for g in ctxs:
            g.destroy()


def test_gauss_invalid_inputs(micsa):
    L, ns, nr = 4, 2, 2
    N = L ** 3
    with pytest.raises(micsa.MicsaError):
        micsa.GaussMicSA(5, 1, 1, 1)
    with micsa.GaussMicSA(L, ns, nr, 1) as g:
        s0, n0, J0 = g.get_state()
        bad = s0.copy(); bad[0, 0, 3] = 0
        with pytest.raises(micsa.MicsaError):
            g.set_state(bad, None)
        badn = np.ones((ns, nr, N)); badn[1, 1, 2] = -1e-9
        with pytest.raises(micsa.MicsaError):
            g.set_state(None, badn)
        badJ = np.zeros((ns, 3, N)); badJ[0, 0, 0] = np.nan
        with pytest.raises(micsa.MicsaError):
            g.set_couplings(badJ)
        for T in (0.0, -1.0, float("nan"), float("inf")):
            with pytest.raises(micsa.MicsaError):
                g.refresh(T, 0)
        with pytest.raises(micsa.MicsaError):
            g.sweep(-1)
        with pytest.raises(micsa.MicsaError):
            g.wander(3, 1, 0)
        gs, gn, gJ = g.get_state()
        np.testing.assert_array_equal(gs, s0); np.testing.assert_array_equal(gn, n0); np.testing.assert_array_equal(gJ, J0)
    with micsa.GaussMicSA(L, ns, 1, 1) as g1:
        assert g1.measure()[2].size == 0
