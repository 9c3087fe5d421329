"""Guard bands around the workspace (-m gpu).  compute-sanitizer cannot be used on this GPU pool, so out-of-range
writes are looked for directly: the library is given a workspace in the middle of a larger buffer filled with a
pattern, a run exercises every kernel family, and the bands on both sides must come back untouched.  (Reads out of
range are caught by the bit-exact parity tests: what is read wrong gives wrong bits.)"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GUARD = 1 << 20          # bytes on each side
PATTERN = 0xA5


def _guarded(micsa, L, ns, nr, seed, sample_offset=0):
    """A MicSA object whose workspace sits between two guard bands of a torch buffer."""
    import torch
    nbytes = micsa.workspace_bytes(L, ns, nr)
    buf = torch.full((nbytes + 2 * GUARD + 256,), PATTERN, dtype=torch.uint8, device="cuda")
    base = (buf.data_ptr() + GUARD + 255) // 256 * 256
    g = object.__new__(micsa.MicSA)
    g.L, g.n_samples, g.n_replicas, g.N = L, ns, nr, L ** 3
    g.n_sys, g.n_pairs, g.seed = ns * nr, ns * (nr * (nr - 1) // 2), seed
    g._ws, g._stream = buf, torch.cuda.current_stream()
    h = micsa._lib.micsa_create_ex(L, ns, nr, seed, sample_offset, ctypes.c_void_p(base), nbytes,
                                   ctypes.c_void_p(g._stream.cuda_stream))
    assert h, micsa.last_error()
    g._h = ctypes.c_void_p(h)
    lo = base - buf.data_ptr()
    return g, buf, lo, lo + nbytes


def _bands_intact(buf, lo, hi):
    import torch
    torch.cuda.synchronize()
    return bool((buf[:lo] == PATTERN).all().item()) and bool((buf[hi:] == PATTERN).all().item())


@pytest.mark.parametrize("L,ns,nr", [(8, 1, 2), (8, 37, 2), (6, 5, 3), (10, 33, 1), (16, 20, 2), (24, 3, 2), (32, 6, 2),
                                     (36, 9, 2), (40, 17, 1), (80, 3, 2)])
def test_no_kernel_writes_outside_the_workspace(micsa, L, ns, nr):
    g, buf, lo, hi = _guarded(micsa, L, ns, nr, 91)
    try:
        assert _bands_intact(buf, lo, hi)                      # create: the Philox start
        sched = [(1.5, 3, 1), (1.1, 2, 2), (0.7, 4, 0)]
        for small in (1, 0):
            g.set_tuning("small_path", small)
            g.anneal(sched, step0=7)
            g.prefetch_refresh(0.9, 30); g.sweep(2); g.refresh_demons(0.9, 30)
            g.sweep_measure(3); g.measure_end(); g.measure_i64()
            g.half_sweep(1); g.half_sweep(0)
            assert _bands_intact(buf, lo, hi), f"small_path={small}"
        for tune in ({"sweep_kernel": 1}, {"sweep_kernel": 2, "pipe_planes": 4}, {"pipe_planes": 1, "pipe_rows": 8}, {"pipe_rows": 4}):
            for k, v in tune.items():
                g.set_tuning(k, v)
            g.sweep(2); g.sweep_measure(1); g.measure_end()
        assert _bands_intact(buf, lo, hi), "sweep kernels"
        g.set_walkers(1); g.sweep(3); g.anneal(sched[:2], step0=50)
        for axis in (0, 1, 2):
            g.wander(axis, +1, 0); g.wander(axis, -1, 1)
        g.set_walkers(0)
        assert _bands_intact(buf, lo, hi), "walkers"
        g.set_gamma(3); g.set_walkers(1); g.anneal(sched[:2], step0=60); g.measure_i64()
        g.set_walkers(0); g.set_gamma(1)
        assert _bands_intact(buf, lo, hi), "gamma"
        g.metropolis_sweep(1.4, 0, 2)
        if nr >= 2:
            g.measure_c4()
        s, m, J = g.get_state()
        g.set_spins(s); g.set_daemons(m); g.set_couplings(J)
        import torch
        row = torch.zeros(g.row_len, dtype=torch.int64, device="cuda")
        g.measure_noalloc(row)
        assert _bands_intact(buf, lo, hi), "metropolis / c4 / state transfer / noalloc"
    finally:
        g.destroy()
