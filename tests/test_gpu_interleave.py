"""Several contexts alive at once, on different streams, with calls interleaved (-m gpu): nothing a context owns
(kernel attributes, side stream, staging, counters, prefetched planes) may leak into another.  Bit-exact against the
oracle driver, which runs every system by itself."""
import numpy as np
import pytest

from oracle import driver

pytestmark = pytest.mark.gpu


def _assert_state(g, s, m, J=None):
    gs, gm, gJ = g.get_state()
    np.testing.assert_array_equal(gs, s)
    np.testing.assert_array_equal(gm, m)
    if J is not None:
        np.testing.assert_array_equal(gJ, J)


def _oracle_state(oracle, L, ns, nr, seed, off=0):
    s = oracle.init_spins(L, ns, nr, seed, sample_offset=off)
    J = oracle.init_bonds(L, ns, seed, sample_offset=off)
    return s, np.zeros_like(s, dtype=np.uint8), J


def test_contexts_on_different_streams_interleaved(micsa, oracle):
    """Four contexts -- general path and small-lattice path, default and high-priority streams -- advanced in turn
    through anneal, single sweeps, prefetched refreshes and both measurement paths."""
    import torch
    specs = [  # L, ns, nr, seed, stream priority (None = the default stream), small_path
        (16, 20, 2, 41, -1, 0), (16, 33, 1, 42, None, 0), (8, 7, 2, 43, -1, 1), (24, 4, 2, 44, 0, 1)]
    ctxs, states, streams = [], [], []
    try:
        for L, ns, nr, seed, prio, small in specs:
            st = torch.cuda.Stream(priority=prio) if prio is not None else None
            g = micsa.MicSA(L, ns, nr, seed, stream=st)
            g.set_tuning("small_path", small)
            ctxs.append(g); streams.append(st); states.append(_oracle_state(oracle, L, ns, nr, seed))
        t_done = [0] * len(specs)
        for rnd in range(3):
            sched = [(1.5 - 0.2 * rnd, 3, 3), (1.4 - 0.2 * rnd, 2, 1)]
            outs = []
            for g in ctxs:                                   # queue everybody's work before anybody is checked
                outs.append(g.anneal(sched, step0=10 * rnd))
            for i, ((L, ns, nr, seed, _, _), g, (s, m, J)) in enumerate(zip(specs, ctxs, states)):
                ref = driver.anneal(L, s, m, J, seed, sched, step0=10 * rnd)
                for k in ("E", "Edem", "Q"):
                    np.testing.assert_array_equal(outs[i][k], ref[k])
                t_done[i] += 5
            # single calls, interleaved: prefetch for all, sweeps for all, then the refreshes
            for g in ctxs:
                g.prefetch_refresh(0.9, 100 + rnd)
            for g in ctxs:
                g.sweep_measure(2)
            rows = [g.measure_end() for g in ctxs]
            for g in ctxs:
                g.refresh_demons(0.9, 100 + rnd)
            for (L, ns, nr, seed, _, _), g, (s, m, J), (E, Ed, Q) in zip(specs, ctxs, states, rows):
                oracle.sweep(L, s, m, J, 2)
                oE, oEd, oQ = oracle.measure(L, s, m, J)
                np.testing.assert_array_equal(E, oE); np.testing.assert_array_equal(Ed, oEd)
                if nr >= 2:
                    np.testing.assert_array_equal(Q, oQ)
                oracle.refresh(L, m, seed, 0.9, 100 + rnd)
                _assert_state(g, s, m, J)
        # one context goes away in the middle; the others carry on
        ctxs[1].destroy()
        for i in (0, 2, 3):
            L, ns, nr, seed, _, _ = specs[i]
            s, m, J = states[i]
            ctxs[i].sweep(3); oracle.sweep(L, s, m, J, 3)
            _assert_state(ctxs[i], s, m, J)
    finally:
        for g in ctxs:
            g.destroy()


def test_same_shape_contexts_share_nothing(micsa, oracle):
    """Two contexts of the same shape and seed but different sample offsets on one stream, calls alternating: the
    staging buffers, counters and prefetched planes are per context."""
    L, ns, nr, seed = 16, 16, 2, 51
    a = micsa.MicSA(L, ns, nr, seed, sample_offset=0)
    b = micsa.MicSA(L, ns, nr, seed, sample_offset=16)
    try:
        sa, sb = _oracle_state(oracle, L, ns, nr, seed, 0), _oracle_state(oracle, L, ns, nr, seed, 16)
        for k in range(3):
            T = 1.2 - 0.3 * k
            a.prefetch_refresh(T, k); b.prefetch_refresh(T + 0.05, k)
            a.sweep(1); b.sweep(2)
            oracle.sweep(L, *sa[:2], sa[2], 1); oracle.sweep(L, *sb[:2], sb[2], 2)
            b.refresh_demons(T + 0.05, k); a.refresh_demons(T, k)
            oracle.refresh(L, sa[1], seed, T, k, 0); oracle.refresh(L, sb[1], seed, T + 0.05, k, 16)
            _assert_state(a, sa[0], sa[1]); _assert_state(b, sb[0], sb[1])
        # set_* of one context between the other's measurement halves
        a.measure_begin()
        b.set_spins(sa[0]); b.set_daemons(sa[1])
        E, Ed, Q = a.measure_end()
        oE, oEd, oQ = oracle.measure(L, sa[0], sa[1], sa[2])
        np.testing.assert_array_equal(E, oE); np.testing.assert_array_equal(Ed, oEd); np.testing.assert_array_equal(Q, oQ)
        _assert_state(b, sa[0], sa[1], sb[2])
    finally:
        a.destroy(); b.destroy()
