"""the N > 1 path (shard by sample, gather rows, max over
ranks) with world_size 2 on CPU over gloo.  No GPU here, so each rank runs the
ORACLE on its shard with its global sample offset; the gathered rows must equal
the unsharded oracle run bit for bit -- which is the property the CUDA library
relies on (tests/test_gpu_parity.py checks the same on the device)."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

L, NS_PER_RANK, NR, SEED = 6, 32, 2, 9
SCHED = [(1.5, 3, 1), (0.9, 2, 2)]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    import oracle
    from oracle import driver
    from paper_2506_16240_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        off = sharding.sample_offset(rank, NS_PER_RANK)
        s = oracle.init_spins(L, NS_PER_RANK, NR, SEED, sample_offset=off)
        J = oracle.init_bonds(L, NS_PER_RANK, SEED, sample_offset=off)
        m = np.zeros_like(s, dtype=np.uint8)
        out = driver.anneal(L, s, m, J, SEED, SCHED, sample_offset=off)
        E = sharding.gather_rows(out["E"], NR)
        Q = sharding.gather_rows(out["Q"], 1)
        t = sharding.max_over_ranks(10.0 + rank)
        if rank == 0:
            np.savez(os.path.join(out_dir, "gathered.npz"), E=E, Q=Q, t=t)
    finally:
        dist.destroy_process_group()


def test_two_ranks_reproduce_the_unsharded_run(tmp_path):
    import oracle
    from oracle import driver
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    got = np.load(tmp_path / "gathered.npz")
    ns = world * NS_PER_RANK
    s = oracle.init_spins(L, ns, NR, SEED)
    J = oracle.init_bonds(L, ns, SEED)
    m = np.zeros_like(s, dtype=np.uint8)
    ref = driver.anneal(L, s, m, J, SEED, SCHED)
    np.testing.assert_array_equal(got["E"], ref["E"])
    np.testing.assert_array_equal(got["Q"], ref["Q"])
    assert float(got["t"]) == 11.0          # MAX over ranks of the per-rank time


def test_offsets_must_keep_philox_blocks_whole():
    from paper_2506_16240_b200 import sharding
    assert sharding.sample_offset(3, 64) == 192
    assert sharding.sample_offset(1, 16) == 32 and sharding.sample_offset(0, 16) == 0
    assert sharding.sample_offset(2, 33) == 128
    with pytest.raises(ValueError):
        sharding.sample_offset(-1, 16)
