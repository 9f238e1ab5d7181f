"""Sharding over ranks: a batch of chains by chains, one large lattice by row slabs.

Chains are independent units, so the path shards with NO data-path collective: rank r owns a contiguous range of
global chain indices and tells its context ``shaken_set_chain_offset(first)``, which makes local chain c draw the
random numbers of global chain ``first + c`` (Philox counter word 1).  The result is bit-identical to one big batch.
The only exchange is the gather of the int64 records at the end (``torch.distributed``: gloo on CPU, nccl on GPU).

This module holds host logic only (index arithmetic and the gather); every step of the method runs in libshaken.
"""
from __future__ import annotations

from typing import Sequence, Tuple

import numpy as np


def chain_shard(n_chains: int, world: int, rank: int) -> Tuple[int, int]:
    """(first, count) of the contiguous, balanced range of global chains rank ``rank`` of ``world`` owns.
    The first ``n_chains % world`` ranks get one chain more; counts may be 0 when world > n_chains."""
    if n_chains < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("bad shard request")
    base, extra = divmod(n_chains, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def shard_couplings(J: Sequence[float], q: Sequence[float], world: int, rank: int):
    """The slices of the per-chain coupling arrays that belong to ``rank``."""
    Ja, qa = np.asarray(J, dtype=np.float64), np.asarray(q, dtype=np.float64)
    if Ja.shape != qa.shape or Ja.ndim != 1:
        raise ValueError("J and q must be 1-D arrays of equal length")
    first, count = chain_shard(Ja.shape[0], world, rank)
    return Ja[first:first + count].copy(), qa[first:first + count].copy()


def open_shard(L: int, n_chains: int, seed: int, world: int, rank: int, **kw):
    """A libshaken context for this rank's chains of an ``n_chains`` batch (None if the rank owns no chain)."""
    from . import shaken

    first, count = chain_shard(n_chains, world, rank)
    if count == 0:
        return None
    s = shaken.Shaken(L, count, seed, **kw)
    s.set_chain_offset(first)
    return s


def gather_records(local: np.ndarray, n_chains: int, group=None, device=None) -> np.ndarray:
    """All-gather per-rank records ``[n_rec, count_r, 6]`` (int64) into ``[n_rec, n_chains, 6]`` in global chain
    order on every rank.  Ranks may own different numbers of chains (including none); shards are padded to the
    largest count for the collective and trimmed afterwards."""
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    first, count = chain_shard(n_chains, world, rank)
    loc = np.ascontiguousarray(local, dtype=np.int64)
    if loc.ndim != 3 or loc.shape[1] != count or loc.shape[2] != 6:
        raise ValueError(f"rank {rank}: records of shape {loc.shape}, expected [n_rec, {count}, 6]")
    n_rec = loc.shape[0]
    width = max(chain_shard(n_chains, world, r)[1] for r in range(world))
    pad = torch.zeros((n_rec, width, 6), dtype=torch.int64)
    pad[:, :count] = torch.from_numpy(loc)
    if device is not None:
        pad = pad.to(device)
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = np.empty((n_rec, n_chains, 6), dtype=np.int64)
    for r, part in enumerate(parts):
        f, c = chain_shard(n_chains, world, r)
        out[:, f:f + c] = part[:, :c].cpu().numpy()
    return out


# ---------------------------------------------------------------------------------------------------------------------
# Row slabs of ONE lattice (second bullet).  Rank r owns a contiguous block of rows; per full step it sends
# its bottom sigma row to the rank below and its top sigma row to the rank above (one exchange, 2 x L bytes) -- the tau row
# just above a slab is redrawn redundantly by that slab, which the counter-based generator makes bit-identical.  On GPUs
# the rows travel by peer stores inside libshaken's kernels (kernel_slab.cuh); this module only does the index
# arithmetic, the exchange of the IPC handles and the final sum of the per-slab int64 records.
# ---------------------------------------------------------------------------------------------------------------------
def slab_shard(L: int, world: int, rank: int) -> Tuple[int, int]:
    """(row0, n_rows) of rank ``rank``: contiguous, balanced, at least two rows each (the library's minimum)."""
    if world < 1 or not 0 <= rank < world or L < 2 * world:
        raise ValueError("bad slab request: every rank needs at least two rows")
    base, extra = divmod(L, world)
    row0 = rank * base + min(rank, extra)
    return row0, base + (1 if rank < extra else 0)


def slab_neighbours(world: int, rank: int) -> Tuple[int, int]:
    """(rank below, rank above) on the torus: the owners of row row0 - 1 and of row row0 + n_rows."""
    return (rank - 1) % world, (rank + 1) % world


def open_slab(L: int, seed: int, world: int, rank: int, **kw):
    """This rank's slab context of an L x L lattice split over ``world`` ranks."""
    from . import shaken

    row0, n_rows = slab_shard(L, world, rank)
    return shaken.ShakenSlab(L, row0, n_rows, seed, **kw)


def connect_slabs_ipc(slab, group=None):
    """Exchange the CUDA IPC handles of the slabs' inboxes over torch.distributed (one process per GPU) and connect every
    slab to its two neighbours.  With a single rank the slab is its own neighbour on both sides (no IPC needed)."""
    import torch.distributed as dist

    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    if world == 1:
        ptr = slab.inbox()
        slab.connect(ptr, ptr)
        return
    handles = [None] * world
    dist.all_gather_object(handles, slab.ipc_export(), group=group)
    below, above = slab_neighbours(world, rank)
    slab.ipc_connect(handles[below], handles[above])


def sum_slab_records(local: np.ndarray, group=None, device=None) -> np.ndarray:
    """The records of the whole lattice: the element-wise sum of the per-slab records ``[n_rec, 1, 6]`` (int64)."""
    import torch
    import torch.distributed as dist

    t = torch.from_numpy(np.ascontiguousarray(local, dtype=np.int64).copy())
    if device is not None:
        t = t.to(device)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t.cpu().numpy()
