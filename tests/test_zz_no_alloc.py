"""micsa_measure_noalloc (include/micsa.h): the measurement with its scratch in the library's static device array
against the existing path (micsa_measure_i64) and the oracle (-m gpu).  Integer sums: bit-exact.

Collected last on purpose (pytest -x); passes alone in a fresh process and after the other tests:
the array is shared by every context of the process and each call clears what it uses.
"""
import numpy as np
import pytest

from micsa_workloads import random_levels, random_pm1

pytestmark = pytest.mark.gpu


def _rows(g, row):
    import torch
    torch.cuda.synchronize()
    r = row.cpu().numpy()
    n = g.n_sys
    return r[:n], r[n:2 * n], r[2 * n:g.row_len]


# (L, n_samples, n_replicas, gamma): pair in a word, ragged lanes, pairs across words (count_xor), one replica,
# several daemon families (count_levels), odd L/2 (V = 1 kernels)
SHAPES = [(16, 20, 2, 1), (8, 37, 2, 1), (6, 5, 3, 1), (8, 40, 1, 1), (8, 9, 2, 3), (10, 3, 4, 2)]


@pytest.mark.parametrize("L,ns,nr,gamma", SHAPES)
def test_measure_noalloc_equals_existing_path(micsa, oracle, L, ns, nr, gamma):
    import torch
    N = L ** 3
    s, J = random_pm1((ns, nr, N), 71), random_pm1((ns, 3, N), 72)
    m = [random_levels((ns, nr, N), 73 + a) for a in range(gamma)]
    with micsa.MicSA(L, ns, nr, 7) as g:
        g.set_gamma(gamma)
        g.set_spins(s); g.set_couplings(J)
        for a in range(gamma):
            g.select_daemon_set(a); g.set_daemons(m[a])
        row = torch.full((g.row_len + 3,), -12345, dtype=torch.int64, device="cuda")   # allocated once, before the calls
        row2 = torch.full((g.row_len,), -777, dtype=torch.int64, device="cuda")
        # two calls in a row, then the existing path on the same state
        g.measure_noalloc(row); g.measure_noalloc(row2)
        E, Ed, Q = g.measure_i64()
        for r in (row, row2):
            nE, nEd, nQ = _rows(g, r)
            np.testing.assert_array_equal(nE, E); np.testing.assert_array_equal(nEd, Ed); np.testing.assert_array_equal(nQ, Q)
        assert (row[g.row_len:].cpu().numpy() == -12345).all()                   # nothing written past the row
        # ... and the oracle
        oE, _, oQ = oracle.measure(L, s, m[0], J)
        oEd = sum(oracle.measure(L, s, m[a], J)[1] for a in range(gamma))
        np.testing.assert_array_equal(E, oE); np.testing.assert_array_equal(Ed, oEd)
        if nr >= 2:
            np.testing.assert_array_equal(Q, oQ)
        # the state moves on; both paths again, the new one first and last (its scratch is not the context's)
        g.refresh_demons(1.1, 3); g.sweep(2)
        g.measure_noalloc(row)
        E, Ed, Q = g.measure_i64()
        g.measure_noalloc(row2)
        for r in (row, row2):
            nE, nEd, nQ = _rows(g, r)
            np.testing.assert_array_equal(nE, E); np.testing.assert_array_equal(nEd, Ed); np.testing.assert_array_equal(nQ, Q)
        # the fused measuring sweep (which uses the context's own counters) is not disturbed
        g.sweep_measure(1)
        fE, fEd, fQ = g.measure_end()
        g.measure_noalloc(row)
        nE, nEd, nQ = _rows(g, row)
        np.testing.assert_array_equal(nE, fE); np.testing.assert_array_equal(nEd, fEd); np.testing.assert_array_equal(nQ, fQ)


def test_measure_noalloc_two_contexts_share_the_scratch(micsa):
    """Calls of different contexts on one stream follow each other on the GPU: each clears what it uses."""
    import torch
    with micsa.MicSA(16, 64, 2, 3) as a, micsa.MicSA(8, 5, 2, 4) as b:
        a.refresh_demons(2.0, 0); b.refresh_demons(0.5, 0)
        ra = torch.zeros(a.row_len, dtype=torch.int64, device="cuda")
        rb = torch.zeros(b.row_len, dtype=torch.int64, device="cuda")
        for _ in range(3):
            a.sweep(1); b.sweep(1)
            a.measure_noalloc(ra); b.measure_noalloc(rb); a.measure_noalloc(ra)
            for g, r in ((a, ra), (b, rb)):
                E, Ed, Q = g.measure_i64()
                nE, nEd, nQ = _rows(g, r)
                np.testing.assert_array_equal(nE, E); np.testing.assert_array_equal(nEd, Ed); np.testing.assert_array_equal(nQ, Q)


def test_measure_noalloc_limits(micsa):
    import torch
    # 257 word lattices need 257 * 64 counters > MICSA_NOALLOC_MAX_COUNTERS = 16384: refused, nothing launched
    with micsa.MicSA(2, 257 * 32, 1, 1) as g:
        row = torch.full((g.row_len,), 5, dtype=torch.int64, device="cuda")
        launches = g.layout_info()["launches"]
        with pytest.raises(micsa.MicsaError, match="MICSA_NOALLOC_MAX_COUNTERS"):
            g.measure_noalloc(row)
        assert g.layout_info()["launches"] == launches
        torch.cuda.synchronize()
        assert (row.cpu().numpy() == 5).all()
        E, Ed, _ = g.measure_i64()                       # the existing path still serves it
        assert E.shape == (257 * 32,) and (Ed == 0).all()
    # 256 word lattices are exactly the limit
    with micsa.MicSA(2, 256 * 32, 1, 1) as g:
        row = torch.zeros(g.row_len, dtype=torch.int64, device="cuda")
        g.measure_noalloc(row)
        E, Ed, Q = g.measure_i64()
        nE, nEd, _ = _rows(g, row)
        np.testing.assert_array_equal(nE, E); np.testing.assert_array_equal(nEd, Ed)
    with micsa.MicSA(4, 2, 2, 1) as g:
        with pytest.raises(micsa.MicsaError):
            g.measure_noalloc(0)                                                  # null
        with pytest.raises(micsa.MicsaError):
            g.measure_noalloc(torch.zeros(g.row_len - 1, dtype=torch.int64, device="cuda"))
        with pytest.raises(micsa.MicsaError):
            g.measure_noalloc(torch.zeros(g.row_len, dtype=torch.int32, device="cuda"))
        host = np.zeros(g.row_len, np.int64)
        with pytest.raises(micsa.MicsaError, match="device"):
            g.measure_noalloc(int(host.ctypes.data))                              # pageable host memory is refused
