"""Pins for the oracle's alternate (even sites / odd sites) parallel heat bath on the square lattice
(SURVEY 8(f) rank 3).  CPU only.

What fixes it from outside the oracle:
  * thresholds: the closed form 1/(1+e^{-2h}) and the exact mirror symmetry;
  * J = 0: every redrawn spin is the top bit of its Philox word -- pins which word a site draws and which sites move;
  * J large: the deterministic majority rule written with numpy rolls (geometry, torus wrap, colours);
  * the theorem the paper quotes (:276, Theorem 2.2 of its ref. [2]): the Gibbs measure of the square-lattice Ising model
    is stationary -- exactly, by enumeration of the 2^16 states of the 4 x 4 torus with the oracle's thresholds, and
    statistically, for long runs of the oracle against the enumerated Gibbs expectations;
  * the global spin flip with complemented random words is an exact symmetry;
  * coupled chains keep their order (attractive dynamics), and coalescence is the first agreement.
"""
import math

import numpy as np
import pytest

from oracle import shaken_oracle as so


def _words_of_colour(L, seed, chain, t, half):
    """rnd of every site of colour `half` from the pinned Philox: the m-th site of the colour in row-major order draws
    word m & 3 of counter (m >> 2, chain, g lo, g hi), g = 2t + half."""
    g = 2 * t + half
    out = np.zeros((L, L), dtype=np.uint64)
    m = 0
    for r in range(L):
        for c in range(L):
            if (r + c) % 2 != half:
                continue
            w = so.philox4x32_10([m >> 2, chain, g & 0xFFFFFFFF, g >> 32], [seed & 0xFFFFFFFF, seed >> 32])
            out[r, c] = int(w[m & 3])
            m += 1
    return out


def test_thresholds_closed_form_and_mirror():
    for J in (0.0, 0.1, 0.4406867935, 0.9, 3.0, 40.0):
        A = so.alt_thresholds(J)
        for k in range(5):
            h = J * (2 * k - 4)                                   # J times the sum of four +-1 neighbours
            want = 2.0**32 / (1.0 + math.exp(-2.0 * h))
            assert abs(int(A[k]) - min(want, 2.0**32 - 1)) <= 1.0
            assert int(A[k]) + int(A[4 - k]) == 2**32             # exact mirror, also when saturated
        assert int(A[2]) == 2**31
        assert all(int(A[k]) <= int(A[k + 1]) for k in range(4))


@pytest.mark.parametrize("L,seed,chain,t", [(4, 5, 0, 0), (6, 2**40 + 3, 2, 7), (10, 9, 1, 2**33)])
def test_J0_spins_are_the_top_bits_of_the_words(L, seed, chain, t):
    rng = np.random.default_rng(L)
    s0 = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
    cur = s0
    for half in (0, 1):
        nxt = so.alt_half_step_rows(cur, seed, chain, 0.0, t, half, 0, L)
        words = _words_of_colour(L, seed, chain, t, half)
        rr, cc = np.indices((L, L))
        active = (rr + cc) % 2 == half
        assert np.array_equal(nxt[active], np.where(words[active] < 2**31, 1, -1))
        assert np.array_equal(nxt[~active], cur[~active])        # the other colour does not move
        cur = nxt


@pytest.mark.parametrize("L", [4, 6, 12])
def test_saturated_J_is_the_majority_rule(L):
    rng = np.random.default_rng(100 + L)
    seed, chain, t = 31, 1, 3
    cur = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
    for half in (0, 1):
        nxt = so.alt_half_step_rows(cur, seed, chain, 30.0, t, half, 0, L)
        field = (np.roll(cur, 1, 0) + np.roll(cur, -1, 0) + np.roll(cur, 1, 1) + np.roll(cur, -1, 1)).astype(int)
        words = _words_of_colour(L, seed, chain, t, half)
        rr, cc = np.indices((L, L))
        active = (rr + cc) % 2 == half
        want = np.where(field > 0, 1, np.where(field < 0, -1, np.where(words < 2**31, 1, -1)))
        want = np.where(active, want, cur)
        assert np.array_equal(nxt, want)
        cur = nxt


def test_row_windows_agree_with_the_whole_lattice():
    L, seed = 8, 77
    rng = np.random.default_rng(8)
    s = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
    whole = so.alt_half_step_rows(s, seed, 0, 0.35, 4, 1, 0, L)
    for r0, n in ((0, 1), (7, 1), (3, 4), (0, 0)):
        assert np.array_equal(so.alt_half_step_rows(s, seed, 0, 0.35, 4, 1, r0, n), whole[r0:r0 + n])


def test_run_is_the_two_half_steps_and_records_are_the_sums():
    L, n_chains, seed, J = 6, 3, 12, np.array([0.2, 0.44, 0.8])
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    start = o.get_spins(0)
    tau0 = o.get_spins(1)
    o.run_alternate(J, 3, 1)
    rec = o.observables()
    assert rec.shape == (3, n_chains, 6)
    for ch in range(n_chains):
        cur = start[ch]
        for t in range(3):
            cur = so.alt_half_step_rows(cur, seed, ch, J[ch], t, 0, 0, L)
            cur = so.alt_half_step_rows(cur, seed, ch, J[ch], t, 1, 0, L)
            s = cur.astype(np.int64)
            assert rec[t, ch, 0] == s.sum()
            assert rec[t, ch, 4] == (s * np.roll(s, -1, 1)).sum() and rec[t, ch, 5] == (s * np.roll(s, -1, 0)).sum()
            assert np.all(rec[t, ch, 1:4] == 0)
        assert np.array_equal(o.get_spins(0)[ch], cur)
    assert np.array_equal(o.get_spins(1), tau0)                  # tau is not part of this dynamics
    assert o.step == 3
    odd = so.Oracle(5, 1, 0)
    with pytest.raises(so.OracleError):
        odd.run_alternate(0.3, 1, 0)                             # odd L: the torus is not bipartite


def _gibbs_4x4(J):
    """All 2^16 states of the 4 x 4 torus: spins [state, site], bond sum, Gibbs weights."""
    L = 4
    n = 1 << (L * L)
    bits = ((np.arange(n)[:, None] >> np.arange(L * L)[None, :]) & 1).astype(np.int8)
    s = (2 * bits - 1).reshape(n, L, L).astype(np.int64)
    bonds = (s * np.roll(s, -1, 2)).sum((1, 2)) + (s * np.roll(s, -1, 1)).sum((1, 2))
    w = np.exp(J * bonds)
    return s, bonds, w / w.sum()


def test_gibbs_measure_is_stationary_exact_enumeration():
    """pi_G P_half = pi_G for both colours, with p(+|k) = A[k] / 2^32 taken from the oracle."""
    J, L = 0.37, 4
    s, _, pi = _gibbs_4x4(J)
    p_plus = so.alt_thresholds(J).astype(np.float64) / 2.0**32
    n = s.shape[0]
    k = ((np.roll(s, 1, 1) + np.roll(s, -1, 1) + np.roll(s, 1, 2) + np.roll(s, -1, 2)) + 4) // 2     # [state, r, c]
    rr, cc = np.indices((L, L))
    weights = 1 << np.arange(L * L).reshape(L, L)
    for half in (0, 1):
        active = (rr + cc) % 2 == half
        # probability that the half-step, from any state with these passive spins, produces the active spins of `state`
        pa = np.where(s == 1, p_plus[k], 1.0 - p_plus[k])
        prod = np.where(active[None], pa, 1.0).prod((1, 2))
        # mass of pi on each passive configuration
        passive_key = (((s + 1) // 2) * np.where(active, 0, weights)[None]).sum((1, 2))
        mass = np.bincount(passive_key, weights=pi, minlength=n)
        pushed = mass[passive_key] * prod
        assert abs(pushed.sum() - 1.0) < 1e-12
        assert np.max(np.abs(pushed - pi)) < 1e-9 * pi.max()


def test_long_runs_sample_the_gibbs_expectations():
    J, L, n_chains = 0.3, 4, 600
    s, bonds, pi = _gibbs_4x4(J)
    e_bonds = float((pi * bonds).sum())
    e_m2 = float((pi * s.sum((1, 2)) ** 2).sum())
    var_bonds = float((pi * bonds**2).sum()) - e_bonds**2
    o = so.Oracle(L, n_chains, 2024)
    o.init(0)
    o.run_alternate(J, 40, 0)                                    # burn-in (tiny lattice, high temperature)
    o.run_alternate(J, 60, 4)                                    # 15 records per chain, 4 steps apart
    rec = o.observables()
    got_bonds = (rec[:, :, 4] + rec[:, :, 5]).astype(np.float64)
    n_eff = n_chains * rec.shape[0] / 2.0                        # allow for some autocorrelation
    assert abs(got_bonds.mean() - e_bonds) < 5.0 * math.sqrt(var_bonds / n_eff), (got_bonds.mean(), e_bonds)
    got_m2 = (rec[:, :, 0].astype(np.float64) ** 2).mean()
    assert abs(got_m2 - e_m2) < 0.06 * e_m2, (got_m2, e_m2)


def test_global_flip_with_complemented_words_is_a_symmetry():
    L, seed, J = 8, 5, 0.41
    a = so.Oracle(L, 2, seed)
    b = so.Oracle(L, 2, seed)
    a.init(0)
    b.set_spins(0, -a.get_spins(0))
    b.set_complement(True)
    a.run_alternate(J, 6, 1)
    b.run_alternate(J, 6, 1)
    assert np.array_equal(a.get_spins(0), -b.get_spins(0))
    ra, rb = a.observables(), b.observables()
    assert np.array_equal(ra[:, :, 0], -rb[:, :, 0]) and np.array_equal(ra[:, :, 4:], rb[:, :, 4:])


def test_coupled_pairs_keep_their_order_and_coalesce():
    L, n_pairs, seed, J, steps = 6, 4, 17, 0.25, 80
    o = so.Oracle(L, 2 * n_pairs, seed)
    o.set_coupling(2)
    o.init(2)
    first_equal = np.full(n_pairs, -1)
    for n in range(1, steps + 1):
        o.run_alternate(J, 1, 0)
        s = o.get_spins(0)
        assert np.all(s[0::2] >= s[1::2])                        # sigma^top >= sigma^bot is preserved
        for g in range(n_pairs):
            if first_equal[g] < 0 and np.array_equal(s[2 * g], s[2 * g + 1]):
                first_equal[g] = n
    assert np.array_equal(o.coalescence(), first_equal)
    assert np.all(first_equal > 0)
    # a pair is the two chains run alone with the leader's random numbers
    alone = so.Oracle(L, 3, seed)                                # chain 2 = leader of pair 1
    alone.init(-1)
    alone.run_alternate(J, 5, 0)
    pair = so.Oracle(L, 2 * n_pairs, seed)
    pair.set_coupling(2)
    pair.init(2)
    pair.run_alternate(J, 5, 0)
    assert np.array_equal(pair.get_spins(0)[3], alone.get_spins(0)[2])
