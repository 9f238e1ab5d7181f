"""Pins for the oracle's coupled chains and coalescence times.  CPU only.

The coupling-group code is pinned against what already stands on its own pins: a group of two coupled chains must be
exactly two UNCOUPLED single-chain runs that happen to use the same seed and chain index (the same sequence of random
numbers), and its coalescence time must be the first step at which those two runs agree, found here
with numpy.  At J = 0 the sites decouple and the coalescence time has a closed-form distribution.
"""
import math

import numpy as np
import pytest

from oracle import shaken_oracle as so


def _pair_by_two_uncoupled_runs(L, seed, leader, J, q, steps):
    """sigma^top from all +1 and sigma^bot from all -1 as two independent contexts with identical randomness."""
    def chain_alone(start):
        o = so.Oracle(L, leader + 1, seed)            # chain index `leader` of a batch == that chain alone (pinned)
        o.init(start)
        out = []
        for _ in range(steps):
            o.run(J, q, 1, 0)
            out.append((o.get_spins(0)[leader].copy(), o.get_spins(1)[leader].copy()))
        return out
    return chain_alone(1), chain_alone(-1)


@pytest.mark.parametrize("L,J,q,seed", [(6, 0.3, 0.4, 3), (8, 0.44, 1.5, 9), (5, 0.7, 0.2, 21)])
def test_group_of_two_is_two_uncoupled_runs_with_the_same_random_numbers(L, J, q, seed):
    steps, n_groups = 60, 3
    o = so.Oracle(L, 2 * n_groups, seed)
    o.set_coupling(2)
    o.init(2)                                          # sandwich start: top all +1, bottom all -1
    assert np.all(o.get_spins(0)[0::2] == 1) and np.all(o.get_spins(0)[1::2] == -1)
    traj = []
    for _ in range(steps):
        o.run(J, q, 1, 0)
        traj.append(o.get_spins(0).copy())
    coal = o.coalescence()
    for g in range(n_groups):
        top, bot = _pair_by_two_uncoupled_runs(L, seed, 2 * g, J, q, steps)
        first_equal = -1
        for n in range(steps):
            assert np.array_equal(traj[n][2 * g], top[n][0]) and np.array_equal(traj[n][2 * g + 1], bot[n][0])
            assert np.all(top[n][0] >= bot[n][0]) and np.all(top[n][1] >= bot[n][1])   # ordering is preserved (:238)
            if first_equal < 0 and np.array_equal(top[n][0], bot[n][0]):
                first_equal = n + 1                    # T = min{n : X_n = Y_n} in full steps
        assert coal[g] == first_equal
        if first_equal > 0:                            # "X_n = Y_n for all n > T"
            assert all(np.array_equal(top[n][0], bot[n][0]) for n in range(first_equal - 1, steps))


def test_coalescence_bookkeeping():
    o = so.Oracle(4, 6, 1)
    assert o.coalescence().size == 0                   # uncoupled: nothing to report
    with pytest.raises(so.OracleError):
        o.set_coupling(4)                              # must divide n_chains
    o.set_coupling(3)
    o.init(2)
    s = o.get_spins(0)
    assert np.all(s[[0, 3]] == 1) and np.all(s[[1, 2, 4, 5]] == -1)
    assert np.all(o.coalescence() == -1)
    o.run(0.0, 20.0, 5, 0)                             # frozen: q saturated, every chain keeps its start
    assert np.all(o.coalescence() == -1)
    o.init(1)                                          # all chains equal from the start: coalesced after one step
    o.run(0.2, 0.3, 2, 0)
    assert np.all(o.coalescence() == 1)
    o.init(2)
    assert np.all(o.coalescence() == -1)               # init forgets


def test_J0_coalescence_time_has_the_closed_form_distribution():
    """J = 0: sites are independent.  In one half-step the two copies of a site (top +, bottom -) draw the same word
    r and disagree afterwards iff T(-q) <= r < T(q): probability rho = (T(q) - T(-q)) / 2^32.  A site is still split
    after n full steps with probability rho^(2n); T = max over the N = L^2 sites, so P(T <= n) = (1 - rho^(2n))^N."""
    L, q, n_groups, seed = 4, 0.35, 3000, 77
    T = so.thresholds(0.0, q)
    rho = (int(T[1]) - int(T[0])) / 2.0**32            # idx 2k+c with k irrelevant at J=0: T[0] = T(-q), T[1] = T(q)
    assert abs(rho - math.tanh(q)) < 1e-8
    o = so.Oracle(L, 2 * n_groups, seed)
    o.set_coupling(2)
    o.init(2)
    o.run(0.0, q, 40, 0)
    coal = o.coalescence()
    assert np.all(coal > 0)
    N = L * L
    cdf = lambda n: (1.0 - rho ** (2 * n)) ** N
    # chi-square over the bins T = 1, 2, ..., 8 and T >= 9
    edges = list(range(1, 9))
    expected = [n_groups * (cdf(n) - cdf(n - 1)) for n in edges] + [n_groups * (1.0 - cdf(8))]
    observed = [int(np.sum(coal == n)) for n in edges] + [int(np.sum(coal >= 9))]
    chi2 = sum((a - b) ** 2 / b for a, b in zip(observed, expected) if b > 5)
    dof = sum(1 for b in expected if b > 5) - 1
    assert chi2 < dof + 5.0 * math.sqrt(2.0 * dof), (chi2, dof, observed, expected)
