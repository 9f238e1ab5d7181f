"""Exact sampling from the stationary measure of the shaken dynamics by coupling from the past.

PAPER.md:240: "it is possible to perform an unbiased sampling from the equilibrium distribution of a Markov chain using
the Propp-Wilson algorithm ... which requires two copies of the Markov chain to be run with the same update function
and the same sequence of random numbers"; :276: "samples are drawn using the Propp-Wilson algorithm".

This is a host driver only: every step runs in libshaken (coupled pairs, sandwich start, fused coalescence test).
What makes it short is the counter-based generator: the random numbers of a full step are a fixed function of its
global index, so "reuse the randomness of times -T .. -1 when restarting from -2T" is just `step = base - 2T`.
"""
from __future__ import annotations

import numpy as np

from . import shaken


def propp_wilson(s: "shaken.Shaken", J, q=None, base: int = 1 << 40, max_doublings: int = 40):
    """One exact draw of sigma per coupling pair of ``s`` (``s.set_coupling(2)`` must have been called; chains 2k and
    2k+1 are the top and bottom copies of pair k and must be given the same couplings).

    For T = 1, 2, 4, ...: both copies start at time -T (top all +1, bottom all -1), the update from time
    t to t+1 uses the random numbers of full-step index ``base + t``, and the pair is done when the copies agree at
    time 0.  All pairs share T; it doubles until the last pair has coalesced.  Different ``base`` values (at least the
    final T apart) or different seeds give independent draws.

    ``q=None`` draws from the alternate (even sites / odd sites) heat bath on the square lattice instead, whose
    stationary measure is the square-lattice Gibbs measure itself (it is attractive too, so the same
    sandwich argument holds).

    Returns (samples [n_pairs, L, L] int8, T)."""
    if getattr(s, "group", 1) != 2:
        raise ValueError("propp_wilson needs coupling groups of two: call set_coupling(2) first")
    Ja = np.ascontiguousarray(J, dtype=np.float64)
    qa = Ja if q is None else np.ascontiguousarray(q, dtype=np.float64)
    if Ja.shape != (s.n_chains,) or qa.shape != (s.n_chains,):
        raise ValueError("J and q must have one entry per chain")
    if not (np.array_equal(Ja[0::2], Ja[1::2]) and np.array_equal(qa[0::2], qa[1::2])):
        raise ValueError("the two copies of a pair must have the same couplings")
    T = 1
    for _ in range(max_doublings):
        if base - T < 0:
            raise ValueError("base is too small for this look-back")
        s.init(shaken.INIT_SANDWICH)     # resets the step counter, so the starting time is set afterwards
        s.step = base - T
        if q is None:
            s.run_alternate(Ja, T, 0)
        else:
            s.run_grid(Ja, qa, T, 0)
        if np.all(s.coalescence() >= 0):
            return s.get_spins(0)[0::2].copy(), T
        T *= 2
    raise RuntimeError("no coalescence within the allowed number of doublings")
