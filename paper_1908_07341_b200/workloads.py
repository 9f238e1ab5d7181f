"""Seeded synthetic workloads shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: it only names lattice sizes, seeds, couplings,
start configurations and step counts.  Both the oracle (oracle/) and the CUDA library receive the
same doubles from here; neither imports the other.

The five configurations are BASELINE.json's ``configs``.  They stand in for
the paper's own workloads: the 200x200 (q,J) grid scan, the 32x32 coalescence runs
(:242), the 512x512 snapshots (:437) and the benchmark sweep at J=0.44, q=0.66 (:441) -- the paper
uses no dataset, every input is a start configuration (all -1 :200, all +1 / all -1 :238) plus
couplings, so the stand-in is exact in kind.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List

import numpy as np

INIT_ALL_UP = 1
INIT_ALL_DOWN = -1
INIT_IID = 0


def critical_J(q: float) -> float:
    """Critical curve J_c(q) = atanh(sqrt(tanh^2 q + 1) - tanh q), eq. (12)."""
    t = math.tanh(q)
    return math.atanh(math.sqrt(t * t + 1.0) - t)


@dataclass
class Workload:
    name: str
    L: int
    n_chains: int
    seed: int
    init: int
    n_steps: int
    obs_every: int
    packed: bool
    J: List[float] = field(default_factory=list)  # one per chain
    q: List[float] = field(default_factory=list)
    burn_in: int = 0  # records dropped by the caller before computing statistics
    note: str = ""

    @property
    def n_sites(self) -> int:
        return self.L * self.L

    @property
    def updates(self) -> int:
        """Site updates of the whole workload: 2 half-steps per full step."""
        return 2 * self.n_steps * self.n_chains * self.n_sites

    def J_array(self) -> np.ndarray:
        return np.asarray(self.J, dtype=np.float64)

    def q_array(self) -> np.ndarray:
        return np.asarray(self.q, dtype=np.float64)

    def scaled(self, n_steps: int | None = None, L: int | None = None) -> "Workload":
        """Same recipe at a reduced step count and/or lattice size (for the oracle's time budget)."""
        w = Workload(**{**self.__dict__})
        if n_steps is not None:
            w.n_steps = int(n_steps)
        if L is not None:
            w.L = int(L)
        w.name = f"{self.name}[L={w.L},steps={w.n_steps}]"
        return w


def grid_couplings():
    """cfg 3 grid: q in {0.1,0.2,0.5,1,2,5,10,20} x J in linspace(0.05,1.2,16) x 4 replicas.
    chain = (iq*16 + iJ)*4 + replica; J_k = 0.05 + k*(1.15/15) in double (SURVEY 8(c) point 17)."""
    qs = [0.1, 0.2, 0.5, 1.0, 2.0, 5.0, 10.0, 20.0]
    Js = [0.05 + k * (1.15 / 15.0) for k in range(16)]
    J, q = [], []
    for iq in range(8):
        for iJ in range(16):
            for _ in range(4):
                J.append(Js[iJ])
                q.append(qs[iq])
    return J, q


def config(i: int) -> Workload:
    """BASELINE.json configs[i-1], i = 1..5."""
    if i == 1:
        return Workload("cfg1", 64, 1, 1, INIT_IID, 1000, 1, False, [0.5], [0.5])
    if i == 2:
        return Workload("cfg2", 1024, 1, 7, INIT_ALL_UP, 10_000, 10, False, [0.6585], [0.6585],
                        note="honeycomb critical point J=q=0.6585 (PAPER.md:151)")
    if i == 3:
        J, q = grid_couplings()
        return Workload("cfg3", 512, 512, 11, INIT_IID, 5000, 1, False, J, q, burn_in=1000,
                        note="(q,J) grid scan, 8 x 16 x 4 replicas (stands in for PAPER.md:200)")
    if i == 4:
        return Workload("cfg4", 16384, 1, 3, INIT_ALL_UP, 1000, 1, False, [0.7], [0.7],
                        note="headline metric: int8, all six sums fused every step")
    if i == 5:
        return Workload("cfg5", 32768, 1, 5, INIT_IID, 500, 1, True, [0.45], [10.0],
                        note="bit-packed multispin, 32 spins per uint32")
    raise ValueError(i)


def paper_benchmark_point(L: int) -> Workload:
    """The paper's own benchmark point (Fig. 20): J=0.44, q=0.66, one update timed."""
    return Workload(f"paper_bench_L{L}", L, 1, 20, INIT_ALL_DOWN, 100, 0, False, [0.44], [0.66])
