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


# ----------------------------------------------------------------------------------------- row slabs of one lattice
SLAB_L, SLAB_STEPS = 24, 4


def test_slab_shard_is_a_partition_with_ring_neighbours():
    for Lx in (16, 24, 100, 16384):
        for world in (1, 2, 3, 8):
            rows = []
            for r in range(world):
                row0, n = parallel.slab_shard(Lx, world, r)
                assert n >= 2
                rows += list(range(row0, row0 + n))
            assert rows == list(range(Lx))
    assert parallel.slab_neighbours(4, 0) == (3, 1) and parallel.slab_neighbours(4, 3) == (2, 0)
    assert parallel.slab_neighbours(1, 0) == (0, 0)
    with pytest.raises(ValueError):
        parallel.slab_shard(6, 4, 0)


def _slab_worker(rank, world, port, out_dir):
    """One rank of the slab plan on CPU.  A rank keeps ONLY its own rows; per full step it sends its bottom sigma row
    down and its top sigma row up (gloo send / recv), redraws the tau row above its slab itself, and never receives a
    tau row.  Rows it does not legitimately hold are poisoned with 0, which the oracle's row function would turn into
    wrong spins if the plan read them."""
    import torch
    import torch.distributed as dist

    from oracle import shaken_oracle as so

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        Lx, J, q = SLAB_L, 0.6, 0.4
        row0, n = parallel.slab_shard(Lx, world, rank)
        below, above = parallel.slab_neighbours(world, rank)
        o = so.Oracle(Lx, 1, SEED)
        o.init(0)
        sigma_own = o.get_spins(0)[0][row0:row0 + n].copy()          # every rank can generate its rows of the iid start
        rec = np.zeros((SLAB_STEPS, 1, 6), dtype=np.int64)
        for t in range(SLAB_STEPS):
            # one exchange per full step: bottom row down, top row up
            bottom, top = torch.from_numpy(sigma_own[0].copy()), torch.from_numpy(sigma_own[-1].copy())
            from_below, from_above = torch.empty(Lx, dtype=torch.int8), torch.empty(Lx, dtype=torch.int8)
            if world == 1:
                from_below, from_above = top.clone(), bottom.clone()
            else:
                reqs = [dist.isend(bottom, below, tag=2 * t), dist.isend(top, above, tag=2 * t + 1),
                        dist.irecv(from_below, below, tag=2 * t + 1), dist.irecv(from_above, above, tag=2 * t)]
                for r in reqs:
                    r.wait()
            src = np.zeros((Lx, Lx), dtype=np.int8)                    # poison
            src[row0:row0 + n] = sigma_own
            src[(row0 - 1) % Lx] = from_below.numpy()
            src[(row0 + n) % Lx] = from_above.numpy()
            # half-step 0: tau rows row0 .. row0 + n (the last one redundantly), from sigma rows row0 - 1 .. row0 + n
            tau = np.zeros((Lx, Lx), dtype=np.int8)
            tau[row0:row0 + n] = so.half_step_rows(src, SEED, 0, J, q, t, 0, row0, n)
            tau[(row0 + n) % Lx] = so.half_step_rows(src, SEED, 0, J, q, t, 0, (row0 + n) % Lx, 1)[0]
            # half-step 1: sigma rows of the slab from tau rows row0 .. row0 + n
            sigma_own = so.half_step_rows(tau, SEED, 0, J, q, t, 1, row0, n)
            # partial sums over the slab's own sites; bonds to the row above use the redundant tau row, bonds to the row
            # below the sigma row received NEXT step -- here taken after one more exchange of the final rows
            full_s = np.zeros((Lx, Lx), dtype=np.int64)
            full_s[row0:row0 + n] = sigma_own
            nb = torch.from_numpy(sigma_own[-1].copy())
            got = torch.empty(Lx, dtype=torch.int8)
            if world == 1:
                got = nb.clone()
            else:
                a, b = dist.isend(nb, above, tag=1000 + t), dist.irecv(got, below, tag=1000 + t)
                a.wait(); b.wait()
            s64, t64 = sigma_own.astype(np.int64), tau[row0:row0 + n].astype(np.int64)
            t_up = np.vstack([tau[row0 + 1:row0 + n], tau[(row0 + n) % Lx][None]]).astype(np.int64)
            s_down = np.vstack([got.numpy()[None], sigma_own[:-1]]).astype(np.int64)
            rec[t, 0] = [s64.sum(), t64.sum(), (s64 * (t_up + np.roll(t64, -1, axis=1))).sum(), (s64 * t64).sum(),
                         (s64 * np.roll(s64, -1, axis=1)).sum(), (s64 * s_down).sum()]
        total = parallel.sum_slab_records(rec)
        np.save(os.path.join(out_dir, f"slab_rec{rank}.npy"), total)
        np.save(os.path.join(out_dir, f"slab_sigma{rank}.npy"), sigma_own)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_ranks_advance_row_slabs_of_one_lattice(tmp_path, world):
    """The slab plan of DESIGN.md section 9 on CPU: one sigma row each way per full step is all that crosses a slab edge,
    and spins and summed records equal the unsplit oracle run bit for bit."""
    import torch.multiprocessing as mp

    from oracle import shaken_oracle as so

    so.build()
    mp.spawn(_slab_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    o = so.Oracle(SLAB_L, 1, SEED)
    o.init(0)
    o.run(0.6, 0.4, SLAB_STEPS, 1)
    want_s, want_r = o.get_spins(0)[0], o.observables()
    for r in range(world):
        row0, n = parallel.slab_shard(SLAB_L, world, r)
        assert np.array_equal(np.load(tmp_path / f"slab_sigma{r}.npy"), want_s[row0:row0 + n]), f"rank {r}: sigma rows differ"
        assert np.array_equal(np.load(tmp_path / f"slab_rec{r}.npy"), want_r), f"rank {r}: summed records differ"
