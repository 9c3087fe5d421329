"""SURVEY.md 8(e) with the PRODUCT on each rank (-m gpu): two processes (gloo rendezvous on 127.0.0.1), each with its
own CUDA context on the box's one GPU and its own shard of samples at its global sample offset, run the schedule through
libmicsa.so, gather the measurement rows and take the MAX of their device times -- the N > 1 plumbing of bench.py
(sharding.sample_offset / gather_rows / max_over_ranks) around the real kernels.  The ranks are independent: no kernel
of one waits for the other (there is no data-path collective to stand in for).  The gathered rows must equal one
unsharded run of the product and the oracle."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu

L, NS_PER_RANK, NR, SEED = 16, 32, 2, 9
SCHED = [(1.5, 3, 1), (0.9, 4, 2)]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    import paper_2506_16240_b200 as micsa
    from paper_2506_16240_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        off = sharding.sample_offset(rank, NS_PER_RANK)
        stream = torch.cuda.Stream()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with micsa.MicSA(L, NS_PER_RANK, NR, SEED, sample_offset=off, stream=stream) as g:
            e0.record(stream)
            out = g.anneal(SCHED)
            e1.record(stream)
            torch.cuda.synchronize()
            spins = g.get_state(daemons=False, couplings=False)[0]
        E = sharding.gather_rows(out["E"], NR)
        Q = sharding.gather_rows(out["Q"], 1)
        t = sharding.max_over_ranks(e0.elapsed_time(e1))
        np.save(os.path.join(out_dir, f"spins{rank}.npy"), spins)
        if rank == 0:
            np.savez(os.path.join(out_dir, "gathered.npz"), E=E, Q=Q, t=t, mine=e0.elapsed_time(e1))
    finally:
        dist.destroy_process_group()


def test_two_ranks_with_the_product(micsa, oracle, tmp_path):
    from oracle import driver
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    got = np.load(tmp_path / "gathered.npz")
    ns = world * NS_PER_RANK
    with micsa.MicSA(L, ns, NR, SEED) as g:
        whole = g.anneal(SCHED)
        ws = g.get_state(daemons=False, couplings=False)[0]
    np.testing.assert_array_equal(got["E"], whole["E"])
    np.testing.assert_array_equal(got["Q"], whole["Q"])
    for rank in range(world):
        np.testing.assert_array_equal(np.load(tmp_path / f"spins{rank}.npy"), ws[rank * NS_PER_RANK:(rank + 1) * NS_PER_RANK])
    s = oracle.init_spins(L, ns, NR, SEED); J = oracle.init_bonds(L, ns, SEED)
    m = np.zeros_like(s, dtype=np.uint8)
    ref = driver.anneal(L, s, m, J, SEED, SCHED)
    np.testing.assert_array_equal(got["E"], ref["E"])
    np.testing.assert_array_equal(ws, s)
    assert float(got["t"]) >= float(got["mine"]) > 0.0       # MAX over ranks of the device times
