"""N > 1 path on CPU: chains sharded over world_size-2 ``gloo`` ranks.

The product cannot run without a GPU, so each rank advances ITS chains with the oracle's per-chain entry point
(``half_step_rows`` takes the GLOBAL chain index, which is what ``shaken_set_chain_offset`` feeds the library's Philox
counter) and the host logic under test -- the shard plan, the coupling slices and the record gather of
``paper_1908_07341_b200.parallel`` -- must reproduce the oracle's single big batch bit for bit on every rank.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1908_07341_b200 import parallel  # noqa: E402

L, N_CHAINS, SEED, STEPS = 16, 5, 23, 3


def _couplings():
    J = np.array([0.2, 0.45, 0.7, 0.05, 1.1])
    q = np.array([0.3, 10.0, 0.7, 2.0, 0.1])
    return J, q


def test_chain_shard_is_a_partition_in_order():
    for n in (0, 1, 5, 512, 513):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                first, count = parallel.chain_shard(n, world, r)
                seen += list(range(first, first + count))
            assert seen == list(range(n))
            counts = [parallel.chain_shard(n, world, r)[1] for r in range(world)]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        parallel.chain_shard(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist

    from oracle import shaken_oracle as so

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        J, q = _couplings()
        first, count = parallel.chain_shard(N_CHAINS, world, rank)
        Jl, ql = parallel.shard_couplings(J, q, world, rank)
        assert Jl.shape == (count,)
        rec = np.zeros((STEPS, count, 6), dtype=np.int64)
        for c in range(count):
            g = first + c                                         # global chain index = counter word 1
            sigma = np.ones((L, L), dtype=np.int8)
            for t in range(STEPS):
                tau = so.half_step_rows(sigma, SEED, g, Jl[c], ql[c], t, 0, 0, L)
                sigma = so.half_step_rows(tau, SEED, g, Jl[c], ql[c], t, 1, 0, L)
                rec[t, c] = so.measure(sigma, tau)
        full = parallel.gather_records(rec, N_CHAINS)
        np.save(os.path.join(out_dir, f"rank{rank}.npy"), full)
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_single_batch(tmp_path):
    import torch.multiprocessing as mp

    from oracle import shaken_oracle as so

    so.build()
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    J, q = _couplings()
    o = so.Oracle(L, N_CHAINS, SEED)
    o.init(1)
    o.run_grid(J, q, STEPS, 1)
    want = o.observables()
    for r in range(world):
        got = np.load(tmp_path / f"rank{r}.npy")
        assert got.shape == want.shape
        assert np.array_equal(got, want), f"rank {r}: gathered records differ from the single-batch oracle"
