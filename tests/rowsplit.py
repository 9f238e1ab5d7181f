"""Test helper: the oracle's row function (oracle.half_step_rows, unchanged) applied to ALL rows of a lattice, the rows
split into bands that run on a thread pool (ctypes releases the GIL during the C call; the oracle's row function only
reads the shared source array).  Legal because a site's random word is a function of (seed, chain, step, half, site)
alone, so bands are independent.  No arithmetic of the method lives here."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from oracle import shaken_oracle as so


def n_threads() -> int:
    return max(1, min(32, os.cpu_count() or 1))


def bands(L: int, parts: int):
    edges = np.linspace(0, L, parts + 1).astype(int)
    return [(int(a), int(b - a)) for a, b in zip(edges[:-1], edges[1:]) if b > a]


def half_step(src: np.ndarray, seed: int, chain: int, J: float, q: float, t: int, half: int, pool=None) -> np.ndarray:
    """The whole target sublattice of one half-step, rows computed band by band in parallel."""
    L = src.shape[-1]
    out = np.empty((L, L), dtype=np.int8)

    def work(b):
        r0, n = b
        out[r0:r0 + n] = so.half_step_rows(src, seed, chain, J, q, t, half, r0, n)

    own = pool is None
    pool = pool or ThreadPoolExecutor(n_threads())
    try:
        list(pool.map(work, bands(L, n_threads() if L * L <= (1 << 22) else 4 * n_threads())))
    finally:
        if own:
            pool.shutdown()
    return out


def mismatching_rows(src: np.ndarray, got: np.ndarray, seed: int, chain: int, J: float, q: float, t: int, half: int, pool=None):
    """Rows of `got` that differ from the oracle's half-step of `src`; compares band by band without building the whole
    expected lattice (L = 65536 is 4.3 GB per layer)."""
    L = src.shape[-1]

    def work(b):
        r0, n = b
        want = so.half_step_rows(src, seed, chain, J, q, t, half, r0, n)
        bad = np.nonzero((want != got[r0:r0 + n]).any(axis=1))[0]
        return [r0 + int(i) for i in bad]

    own = pool is None
    pool = pool or ThreadPoolExecutor(n_threads())
    try:
        res = list(pool.map(work, bands(L, 8 * n_threads())))
    finally:
        if own:
            pool.shutdown()
    return [r for part in res for r in part]
