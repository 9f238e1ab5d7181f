"""Pins for the oracle's diagonal correlation sums.  CPU only."""
import math

import numpy as np

from oracle import shaken_oracle as so


def _random_sigma(L, n, seed):
    rng = np.random.default_rng(seed)
    return np.where(rng.integers(0, 2, size=(n, L, L)) == 1, 1, -1).astype(np.int8)


def test_trivial_values_wrap_and_hand_made_configurations():
    L = 6
    o = so.Oracle(L, 3, 1)
    o.init(1)
    d = o.diag_correlations([0, 1, 2, 5, 6, 7])
    assert np.all(d == L * L)                                    # all +1: every product is +1
    s = _random_sigma(L, 3, 7)
    o.set_spins(0, s)
    d = o.diag_correlations([0, 1, 2, 3, L, L + 1, L + 2])
    assert np.all(d[:, 0, :] == L * L)                           # l = 0: sigma_x^2
    assert np.array_equal(d[:, 4], d[:, 0]) and np.array_equal(d[:, 5], d[:, 1]) and np.array_equal(d[:, 6], d[:, 2])
    # a single -1 at (r, c) = (1, 2) in a sea of +1 flips exactly two products of each sum
    one = np.ones((3, L, L), dtype=np.int8)
    one[:, 1, 2] = -1
    o.set_spins(0, one)
    assert np.all(o.diag_correlations([1, 2]) == L * L - 4)
    # two -1 on one SW-NE diagonal at distance 2, (1,1) and (3,3): their mutual product is +1 again for l = 2 only
    two = np.ones((3, L, L), dtype=np.int8)
    two[:, 1, 1] = -1
    two[:, 3, 3] = -1
    o.set_spins(0, two)
    d = o.diag_correlations([1, 2])
    assert np.all(d[:, 0, 0] == L * L - 8) and np.all(d[:, 1, 0] == L * L - 4) and np.all(d[:, :, 1] == L * L - 8)
    # ... and on one NW-SE diagonal, (3,1) and (1,3)
    two[:] = 1
    two[:, 3, 1] = -1
    two[:, 1, 3] = -1
    o.set_spins(0, two)
    d = o.diag_correlations([1, 2])
    assert np.all(d[:, 1, 1] == L * L - 4) and np.all(d[:, 0, 1] == L * L - 8) and np.all(d[:, :, 0] == L * L - 8)


def test_lattice_symmetries():
    """Transposition keeps both diagonals; mirroring the columns exchanges SW-NE and NW-SE; translations keep both."""
    L, n = 8, 4
    s = _random_sigma(L, n, 11)
    ells = [1, 2, 3, 4]
    o = so.Oracle(L, n, 1)
    o.set_spins(0, s)
    d = o.diag_correlations(ells)
    o.set_spins(0, np.ascontiguousarray(s.transpose(0, 2, 1)))
    assert np.array_equal(o.diag_correlations(ells), d)
    o.set_spins(0, np.ascontiguousarray(s[:, :, ::-1]))
    assert np.array_equal(o.diag_correlations(ells), d[:, :, ::-1])
    o.set_spins(0, np.roll(np.roll(s, 3, axis=1), 5, axis=2))
    assert np.array_equal(o.diag_correlations(ells), d)
    assert not np.array_equal(d[:, :, 0], d[:, :, 1])            # the two diagonals do differ on random input


def test_q0_rings_give_the_textbook_correlations_on_the_nwse_diagonal_only():
    """q = 0: rings of 2L spins run NW-SE, so after equilibration
    <sigma_x sigma_{x + l steps along NW-SE}> = (u^{2l} + u^{2L-2l}) / (1 + u^{2L}), u = tanh J (2l bonds apart on the
    ring), and the SW-NE partner sits on another ring (2l not a multiple of L): 0.  This is also the small-q statement
    of the paper: SW-NE correlations are weaker than NW-SE ones."""
    L, J, n_chains = 6, 0.5, 6000
    u, n = math.tanh(J), 2 * L
    o = so.Oracle(L, n_chains, 321)
    o.init(0)
    o.run(J, 0.0, 40, 0)
    d = o.diag_correlations([1, 2]).astype(np.float64).sum(axis=0) / (n_chains * L * L)
    se = 1 / math.sqrt(n_chains * L * L)
    for i, l in enumerate((1, 2)):
        want = (u ** (2 * l) + u ** (n - 2 * l)) / (1 + u**n)
        assert abs(d[i, 1] - want) < 6 * se, (l, d[i, 1], want)
        assert abs(d[i, 0]) < 6 * se, (l, d[i, 0])
