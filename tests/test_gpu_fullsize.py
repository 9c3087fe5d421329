"""The bit-exact parity protocol of SURVEY.md 8(c) at BASELINE's full sizes (-m gpu).

"Configs 2-5: identical seeds; compare full state after each of the first n
sweeps covering >= 3 refreshes; beyond that, compare the int64 measurement sums
at sparse checkpoints as far as the oracle budget allows, and run P2/P3 on the
GPU for the full length."  What each case compares is listed in DESIGN.md 3.1.

The CUDA path runs the whole configuration in the launch configuration
bench.py times (default kernel selection, prefetched refresh, measurement fused
into the 10th sweep of a group); the oracle runs the same systems (all of them
at config 4, sampled blocks of samples elsewhere -- systems never interact).
"""
import numpy as np
import pytest

from micsa_workloads import CONFIGS, schedule_for
from oracle import driver

pytestmark = pytest.mark.gpu


def _per_sweep_parity(micsa, oracle, cfg, T, interval, n_sweeps, blocks, width, tune=None):
    """State after EVERY sweep (and after every refresh) of the first n_sweeps
    sweeps; measurement sums at the end of every refresh interval."""
    L, nr, seed = cfg.L, cfg.n_replicas, cfg.seed
    ref = []
    for k in blocks:
        s = oracle.init_spins(L, width, nr, seed, sample_offset=k)
        J = oracle.init_bonds(L, width, seed, sample_offset=k)
        ref.append((k, s, np.zeros_like(s, dtype=np.uint8), J))

    from concurrent.futures import ThreadPoolExecutor
    pool = ThreadPoolExecutor(1)

    def compare(g, what, oracle_step):
        # the oracle's step runs on a host thread (its calls release the GIL) while the library's state comes back
        fut = pool.submit(oracle_step)
        gs, gm, _ = g.get_state(couplings=False)
        fut.result()
        for k, s, m, _ in ref:
            # (np.array_equal first: assert_array_equal is several times slower on 131 MB arrays; it writes the report)
            if not np.array_equal(gs[k:k + width], s):
                np.testing.assert_array_equal(gs[k:k + width], s, err_msg=f"spins, samples {k}.., {what}")
            if not np.array_equal(gm[k:k + width], m):
                np.testing.assert_array_equal(gm[k:k + width], m, err_msg=f"daemons, samples {k}.., {what}")

    with micsa.MicSA(L, cfg.n_samples, nr, seed) as g:
        for key, v in (tune or {}).items():
            g.set_tuning(key, v)
        gJ = g.get_state(spins=False, daemons=False)[2]
        for k, _, _, J in ref:
            np.testing.assert_array_equal(gJ[k:k + width], J)
        for t in range(n_sweeps):
            if t % interval == 0:
                r = t // interval
                g.refresh_demons(T, r)
                if t + interval < n_sweeps:
                    g.prefetch_refresh(T, r + 1)          # generated under the sweeps, as bench.py does
                compare(g, f"after refresh {r}", lambda: [oracle.refresh(L, m, seed, T, r, k) for k, _, m, _ in ref])
            last_of_group = (t + 1) % interval == 0
            if last_of_group:
                g.sweep_measure(1)
                E, Ed, Q = g.measure_end()
            else:
                g.sweep(1)
            compare(g, f"after sweep {t + 1}", lambda: [oracle.sweep(L, s, m, J, 1) for _, s, m, J in ref])
            if last_of_group:
                for k, s, m, J in ref:
                    oE, oEd, oQ = oracle.measure(L, s, m, J)
                    sl = slice(k * nr, (k + width) * nr)
                    np.testing.assert_array_equal(E[sl], oE)
                    np.testing.assert_array_equal(Ed[sl], oEd)
                    if nr == 2:
                        np.testing.assert_array_equal(Q[k:k + width], oQ)
    pool.shutdown()


def test_config4_every_sample_every_sweep(micsa, oracle):
    """Config 4, ALL 16 samples x 2 replicas (every lane of the 32-lane word at L = 160): the full state after each
    of the first 30 sweeps and each of their 3 refreshes."""
    cfg = CONFIGS[4]
    _per_sweep_parity(micsa, oracle, cfg, cfg.temperatures[0], 10, 30, blocks=(0,), width=cfg.n_samples)


def test_config4_every_sample_alternative_kernels(micsa, oracle):
    """The same lattice under the non-default sweep kernels (12 sweeps, 2 refreshes, all 32 lanes)."""
    cfg = CONFIGS[4]
    for tune in ({"sweep_kernel": 2, "pipe_planes": 1}, {"sweep_kernel": 1}):
        _per_sweep_parity(micsa, oracle, cfg, cfg.temperatures[0], 6, 12, blocks=(0,), width=cfg.n_samples, tune=tune)


@pytest.mark.parametrize("T", CONFIGS[2].temperatures)
def test_config2_every_sweep(micsa, oracle, T):
    _per_sweep_parity(micsa, oracle, CONFIGS[2], T, 10, 30, blocks=(0, 28, 60), width=4)


@pytest.mark.parametrize("interval,n_sweeps", [(1, 4), (10, 30)])
def test_config3_every_sweep(micsa, oracle, interval, n_sweeps):
    cfg = CONFIGS[3]
    _per_sweep_parity(micsa, oracle, cfg, cfg.temperatures[0], interval, n_sweeps, blocks=(0, 62, 124), width=4)


def test_config3_interval_100(micsa, oracle):
    """Refresh interval 100: 3 refreshes = 300 sweeps on one sample; state after sweeps 1..10 of every interval and
    at its end (the oracle still runs every sweep)."""
    cfg = CONFIGS[3]
    L, nr, seed, T, k = cfg.L, cfg.n_replicas, cfg.seed, cfg.temperatures[0], 77
    s = oracle.init_spins(L, 1, nr, seed, sample_offset=k)
    J = oracle.init_bonds(L, 1, seed, sample_offset=k)
    m = np.zeros_like(s, dtype=np.uint8)
    with micsa.MicSA(L, cfg.n_samples, nr, seed) as g:
        for r in range(3):
            g.refresh_demons(T, r); oracle.refresh(L, m, seed, T, r, k)
            g.prefetch_refresh(T, r + 1)
            for t in range(10):
                g.sweep(1); oracle.sweep(L, s, m, J, 1)
                gs, gm, _ = g.get_state(couplings=False)
                np.testing.assert_array_equal(gs[k:k + 1], s); np.testing.assert_array_equal(gm[k:k + 1], m)
            g.sweep(89); g.sweep_measure(1); E, Ed, Q = g.measure_end()
            oracle.sweep(L, s, m, J, 90)
            gs, gm, _ = g.get_state(couplings=False)
            np.testing.assert_array_equal(gs[k:k + 1], s); np.testing.assert_array_equal(gm[k:k + 1], m)
            oE, oEd, oQ = oracle.measure(L, s, m, J)
            np.testing.assert_array_equal(E[k * nr:(k + 1) * nr], oE)
            np.testing.assert_array_equal(Ed[k * nr:(k + 1) * nr], oEd)
            np.testing.assert_array_equal(Q[k:k + 1], oQ)


def test_config5_every_sweep(micsa, oracle):
    """Config 5 (1024 single-replica samples, 201 MB of state, lattice groups): the first three ramp steps."""
    cfg = CONFIGS[5]
    sched = schedule_for(cfg, n_sweeps=30)
    L, seed = cfg.L, cfg.seed
    blocks, width = (0, 500, 1020), 4
    ref = []
    for k in blocks:
        s = oracle.init_spins(L, width, 1, seed, sample_offset=k)
        ref.append((k, s, np.zeros_like(s, dtype=np.uint8), oracle.init_bonds(L, width, seed, sample_offset=k)))
    with micsa.MicSA(L, cfg.n_samples, 1, seed) as g:
        for r, (T, n, _) in enumerate(sched):
            g.refresh_demons(T, r)
            if r + 1 < len(sched):
                g.prefetch_refresh(sched[r + 1][0], r + 1)
            for k, _, m, _ in ref:
                oracle.refresh(L, m, seed, T, r, k)
            for t in range(n):
                if t == 3:
                    g.sweep(n - 4)                     # a multi-sweep call: goes lattice group by lattice group
                    for _, s, m, J in ref:
                        oracle.sweep(L, s, m, J, n - 4)
                elif t > 3 and t < n - 1:
                    continue
                else:
                    g.sweep(1)
                    for _, s, m, J in ref:
                        oracle.sweep(L, s, m, J, 1)
                gs, gm, _ = g.get_state(couplings=False)
                for k, s, m, _ in ref:
                    np.testing.assert_array_equal(gs[k:k + width], s)
                    np.testing.assert_array_equal(gm[k:k + width], m)
            E, Ed, _ = g.measure_i64()
            for k, s, m, J in ref:
                oE, oEd, _ = oracle.measure(L, s, m, J)
                np.testing.assert_array_equal(E[k:k + width], oE)
                np.testing.assert_array_equal(Ed[k:k + width], oEd)


@pytest.mark.parametrize("walkers", [False, True])
def test_config4_gamma6_full_size(micsa, oracle, walkers):
    """gamma = 6 daemon families / six walkers per spin (Eq. 13) on the L = 160 lattice of config 4
    (238 MB of state; with walkers the exchanges along X, Y and Z ride on the odd half-sweeps): two refreshes, three
    timesteps each = 36 sweeps, sampled samples against the oracle driver -- spins, every family, rows."""
    cfg = CONFIGS[4]
    L, nr, seed, gamma = cfg.L, cfg.n_replicas, cfg.seed, 6
    sched = [(0.9, 3, 1), (0.8, 3, 3)]
    with micsa.MicSA(L, cfg.n_samples, nr, seed) as g:
        g.set_gamma(gamma)
        g.set_walkers(1 if walkers else 0)
        out = g.anneal(sched)
        spins = g.get_state(daemons=False, couplings=False)[0]
        fam = []
        for alpha in range(gamma):
            g.select_daemon_set(alpha)
            fam.append(g.get_state(spins=False, couplings=False)[1])
        assert g.get_time() == 6
    for k in (3, 12):
        s = oracle.init_spins(L, 1, nr, seed, sample_offset=k)
        J = oracle.init_bonds(L, 1, seed, sample_offset=k)
        m = np.zeros((gamma, 1, nr, L ** 3), np.uint8)
        ref = driver.anneal(L, s, m, J, seed, sched, sample_offset=k, walkers=walkers)
        np.testing.assert_array_equal(spins[k:k + 1], s)
        for alpha in range(gamma):
            np.testing.assert_array_equal(fam[alpha][k:k + 1], m[alpha])
        sl = slice(k * nr, (k + 1) * nr)
        np.testing.assert_array_equal(out["E"][:, sl], ref["E"])
        np.testing.assert_array_equal(out["Edem"][:, sl], ref["Edem"])
        np.testing.assert_array_equal(out["Q"][:, k:k + 1], ref["Q"])


def test_config2_late_checkpoint_rows(micsa, oracle):
    """Beyond the per-sweep window: the int64 sums at sweeps 250, 500, 750, 1000 of config 2 (T = 2.0) and the state at
    sweep 1000, four samples against the oracle."""
    cfg = CONFIGS[2]
    L, nr, seed, k, width = cfg.L, cfg.n_replicas, cfg.seed, 36, 4
    sched = schedule_for(cfg, T=2.0, n_sweeps=1000, measure_every=10)
    with micsa.MicSA(L, cfg.n_samples, nr, seed) as g:
        out = g.anneal(sched)
        gs, gm, _ = g.get_state(couplings=False)
    s = oracle.init_spins(L, width, nr, seed, sample_offset=k)
    J = oracle.init_bonds(L, width, seed, sample_offset=k)
    m = np.zeros_like(s, dtype=np.uint8)
    ref = driver.anneal(L, s, m, J, seed, sched, sample_offset=k)
    np.testing.assert_array_equal(gs[k:k + width], s)
    np.testing.assert_array_equal(gm[k:k + width], m)
    sl = slice(k * nr, (k + width) * nr)
    for row in (24, 49, 74, 99):
        assert out["sweep"][row] == ref["sweep"][row] == 10 * (row + 1)
        np.testing.assert_array_equal(out["E"][row, sl], ref["E"][row])
        np.testing.assert_array_equal(out["Edem"][row, sl], ref["Edem"][row])
        np.testing.assert_array_equal(out["Q"][row, k:k + width], ref["Q"][row])


def _full_length_invariants(micsa, cfg, sched_step, n_steps, n_check):
    """P2 / P3 over a run of the configuration's REAL length: n_steps schedule steps through
    micsa_anneal, interrupted at n_check evenly spaced places by a hand-made step (refresh, measure, sweeps, measure)
    in which E + E_daemon must be the same integer before and after the sweeps, in every system; at the end n sweeps
    forward and n with the half-sweeps reversed restore the state."""
    T, n_sw = sched_step
    chunk = n_steps // n_check
    with micsa.MicSA(cfg.L, cfg.n_samples, cfg.n_replicas, cfg.seed) as g:
        done = 0
        for c in range(n_check):
            g.anneal([(T, n_sw, 0)] * (chunk - 1), step0=done, trace=False)
            done += chunk - 1
            g.refresh_demons(T, done)
            E0, Ed0, _ = g.measure_i64()
            g.sweep(n_sw - 1); g.sweep_measure(1)
            E1, Ed1, _ = g.measure_end()
            np.testing.assert_array_equal(E0 + Ed0, E1 + Ed1)
            done += 1
        assert g.counters()["attempts"] == done * n_sw * cfg.attempts_per_sweep
        s0, m0, _ = g.get_state(couplings=False)
        g.sweep(25)
        for _ in range(25):
            g.half_sweep(1); g.half_sweep(0)
        s1, m1, _ = g.get_state(couplings=False)
        np.testing.assert_array_equal(s1, s0)
        np.testing.assert_array_equal(m1, m0)
        return E1 / cfg.N


def test_config4_full_length_invariants(micsa):
    cfg = CONFIGS[4]
    e = _full_length_invariants(micsa, cfg, (cfg.temperatures[0], 10), cfg.n_sweeps // 10, 20)
    assert -1.75 < e.mean() < -1.73                       # -1.7402 after 1e5 sweeps at T = 0.9


def test_config3_full_length_invariants(micsa):
    cfg = CONFIGS[3]
    e = _full_length_invariants(micsa, cfg, (cfg.temperatures[0], 10), cfg.n_sweeps // 10, 20)
    assert -1.77 < e.mean() < -1.75                       # -1.7622 at T = 0.7, R = 10


def test_config5_full_length_invariants(micsa):
    """Config 5's ramp at its real length, E + E_daemon checked inside 20 of its 1000 steps, reversal at T = 0.2."""
    cfg = CONFIGS[5]
    sched = schedule_for(cfg)
    with micsa.MicSA(cfg.L, cfg.n_samples, 1, cfg.seed) as g:
        for c in range(20):
            lo = c * 50
            g.anneal(sched[lo:lo + 49], step0=lo, trace=False)
            T = sched[lo + 49][0]
            g.refresh_demons(T, lo + 49)
            E0, Ed0, _ = g.measure_i64()
            g.sweep(9); g.sweep_measure(1)
            E1, Ed1, _ = g.measure_end()
            np.testing.assert_array_equal(E0 + Ed0, E1 + Ed1)
        assert (E1 / cfg.N).mean() < -1.76                # annealed: -1.7714
        s0, m0, _ = g.get_state(couplings=False)
        g.sweep(20)
        for _ in range(20):
            g.half_sweep(1); g.half_sweep(0)
        s1, m1, _ = g.get_state(couplings=False)
        np.testing.assert_array_equal(s1, s0)
        np.testing.assert_array_equal(m1, m0)


@pytest.mark.parametrize("l2_groups", [1, 0])
def test_table3_shape_sampled(micsa, oracle, l2_groups):
    """The state-larger-than-L2 workload of bench.py's `hbm_resident` record (160^3 x 128 systems, the shape of the
    paper's Table 3; four word lattices, 295 MB): two refresh intervals in the launch configuration
    the bench times (multi-sweep calls lattice group by lattice group, or every half-sweep over all lattices), three
    sampled samples from different word lattices against the oracle -- state, rows, counters."""
    L, ns, nr, seed, T = 160, 64, 2, 4, 0.9
    sched = [(T, 10, 10)] * 2
    with micsa.MicSA(L, ns, nr, seed) as g:
        g.set_tuning("l2_groups", l2_groups)
        assert g.layout_info()["state_bytes"] == 294912000
        out = g.anneal(sched)
        gs, gm, _ = g.get_state(couplings=False)
        assert g.counters()["attempts"] == 20 * L ** 3 * ns * nr
    for k in (0, 17, 63):
        s = oracle.init_spins(L, 1, nr, seed, sample_offset=k); J = oracle.init_bonds(L, 1, seed, sample_offset=k)
        m = np.zeros_like(s, dtype=np.uint8)
        ref = driver.anneal(L, s, m, J, seed, sched, sample_offset=k)
        np.testing.assert_array_equal(gs[k:k + 1], s)
        np.testing.assert_array_equal(gm[k:k + 1], m)
        np.testing.assert_array_equal(out["E"][:, k * nr:(k + 1) * nr], ref["E"])
        np.testing.assert_array_equal(out["Edem"][:, k * nr:(k + 1) * nr], ref["Edem"])
        np.testing.assert_array_equal(out["Q"][:, k:k + 1], ref["Q"])


def test_largest_lattice_offsets_beyond_2_31_bytes(micsa, oracle):
    """Maximum size: L = 1040 (N = 1.125e9 sites, just below the 2^31 limit of the 32-bit site index; a parity array
    holds 2.25 GB, so the kernels' unsigned 32-bit byte offsets go beyond 2^31).  One sample x two replicas: the Philox
    start, one refresh, one sweep, the separate and the fused measurement against the oracle, every site.  About two
    minutes, mostly the oracle; 20 GB of host memory."""
    from concurrent.futures import ThreadPoolExecutor
    L, ns, nr, seed, T = 1040, 1, 2, 3, 0.9
    # the oracle's start, bonds and refresh do not depend on one another: three host threads (the calls release the
    # GIL), the library's own start and first sweep meanwhile
    m = np.zeros((ns, nr, L ** 3), np.uint8)
    with ThreadPoolExecutor(3) as pool, micsa.MicSA(L, ns, nr, seed) as g:
        f_s = pool.submit(oracle.init_spins, L, ns, nr, seed)
        f_J = pool.submit(oracle.init_bonds, L, ns, seed)
        f_m = pool.submit(oracle.refresh, L, m, seed, T, 7)
        gs, gm, gJ = g.get_state()
        g.refresh_demons(T, 7); g.sweep(1)
        s, J = f_s.result(), f_J.result()
        assert np.array_equal(gs, s) and np.array_equal(gJ, J) and not gm.any()
        del gJ, gs, gm
        f_m.result()
        oracle.sweep(L, s, m, J, 1)
        gs, gm, _ = g.get_state(couplings=False)
        assert np.array_equal(gs, s) and np.array_equal(gm, m)
        del gs, gm
        E, Ed, Q = g.measure_i64()
        oE, oEd, oQ = oracle.measure(L, s, m, J)
        np.testing.assert_array_equal(E, oE); np.testing.assert_array_equal(Ed, oEd); np.testing.assert_array_equal(Q, oQ)
        g.sweep_measure(1); E2, Ed2, _ = g.measure_end()
        np.testing.assert_array_equal(E2 + Ed2, E + Ed)           # PAPER.md:124 at this size too
        assert g.counters()["attempts"] == 2 * L ** 3 * ns * nr


@pytest.mark.parametrize("L,ns,nr", [(62, 33, 2), (100, 17, 1), (50, 40, 3), (36, 70, 2)])
def test_lattices_off_the_fast_path_at_medium_size(micsa, oracle, L, ns, nr):
    """L not a multiple of 8 (the kernels with 1 or 2 words per thread; L = 36: 4 words but no pipelined kernel), ragged
    sample counts, 1 / 2 / 3 replicas, at sizes where a plane no longer fits a block: start, two refreshes, sweeps,
    wandering, Metropolis and both measurement paths against the oracle, every site."""
    seed, T = 9, 1.1
    s = oracle.init_spins(L, ns, nr, seed); J = oracle.init_bonds(L, ns, seed)
    m = np.zeros_like(s, dtype=np.uint8)

    def same(g, with_J=False):
        gs, gm, gJ = g.get_state(couplings=with_J)
        assert np.array_equal(gs, s) and np.array_equal(gm, m) and (not with_J or np.array_equal(gJ, J))

    with micsa.MicSA(L, ns, nr, seed) as g:
        same(g, True)
        for r in range(2):
            g.prefetch_refresh(T - 0.3 * r, r); g.refresh_demons(T - 0.3 * r, r); oracle.refresh(L, m, seed, T - 0.3 * r, r)
            g.sweep(2); oracle.sweep(L, s, m, J, 2)
            same(g)
            g.sweep_measure(1); E, Ed, Q = g.measure_end(); oracle.sweep(L, s, m, J, 1)
            oE, oEd, oQ = oracle.measure(L, s, m, J)
            np.testing.assert_array_equal(E, oE); np.testing.assert_array_equal(Ed, oEd)
            if nr >= 2:
                np.testing.assert_array_equal(Q, oQ)
        t0 = g.get_time()
        g.set_walkers(1); g.sweep(3)
        for t in range(3):
            oracle.sweep(L, s, m, J, 1); oracle.wander(L, m, 0, +1, (t0 + t) & 1)
        same(g)
        g.set_walkers(0)
        g.metropolis_sweep(1.3, 5, 2); oracle.metropolis_checkerboard(L, s, J, seed, 1.3, 5, 2)
        same(g)
        E, Ed, Q = g.measure_i64()
        oE, oEd, oQ = oracle.measure(L, s, m, J)
        np.testing.assert_array_equal(E, oE); np.testing.assert_array_equal(Ed, oEd)


def test_full_length_runs_agree_between_the_refresh_modes(micsa):
    """Beyond what the oracle can follow: the same long schedule with the refreshes generated in line (default
    stream) and one step ahead on the side stream (high-priority stream) must leave identical bits -- a race between
    the side stream's writes and the sweeps would show here.  Config 4, 2 000 steps = 20 000 sweeps, rows every 100
    steps; config 2 at its full 10^4 sweeps on the chained small-lattice path against the general path."""
    import torch
    cfg = CONFIGS[4]
    sched = [(cfg.temperatures[0], 10, 10 if (k + 1) % 100 == 0 else 0) for k in range(2000)]
    res = []
    for prio in (None, -1):
        stream = torch.cuda.Stream(priority=prio) if prio is not None else None
        with micsa.MicSA(cfg.L, cfg.n_samples, cfg.n_replicas, cfg.seed, stream=stream) as g:
            out = g.anneal(sched)
            res.append((out, g.get_state(couplings=False)[:2], g.counters()))
    (o0, (s0, m0), c0), (o1, (s1, m1), c1) = res
    assert np.array_equal(s0, s1) and np.array_equal(m0, m1)
    for k in ("sweep", "E", "Edem", "Q"):
        np.testing.assert_array_equal(o0[k], o1[k])
    assert c0 == c1 and o0["E"].shape[0] == 20

    cfg = CONFIGS[2]
    sched = [(2.0, 10, 10 if (k + 1) % 50 == 0 else 0) for k in range(1000)]
    res = []
    for small in (1, 0):
        with micsa.MicSA(cfg.L, cfg.n_samples, cfg.n_replicas, cfg.seed, stream=torch.cuda.Stream(priority=-1)) as g:
            g.set_tuning("small_path", small)
            out = g.anneal(sched)
            res.append((out, g.get_state(couplings=False)[:2], g.counters()))
    (o0, (s0, m0), c0), (o1, (s1, m1), c1) = res
    assert np.array_equal(s0, s1) and np.array_equal(m0, m1)
    for k in ("sweep", "E", "Edem", "Q"):
        np.testing.assert_array_equal(o0[k], o1[k])
    assert c0 == c1 and o0["E"].shape[0] == 20
