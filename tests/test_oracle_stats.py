"""Pins of the oracle's derived statistics and energy (CPU only, eq. 17,
eq. 5 :81-84).  Every expected value below is written out by hand (or is a closed form of the chosen records),
none is computed by either implementation.  Each test names the mistake it would catch."""
import math

import numpy as np

from oracle import shaken_oracle as so


def test_derived_stats_hand_computed_four_records():
    """Records M = (2, -2, 4, 0) on N = 4 sites: m = M/N = (1/2, -1/2, 1, 0).
    <m> = 1/4; <|m|> = 1/2; <m^2> = (1/4 + 1/4 + 1 + 0)/4 = 3/8; <m^4> = (1/16 + 1/16 + 1 + 0)/4 = 9/32;
    Var m = 3/8 - 1/16 = 5/16 (population variance, "average and variance");
    U = 1 - (9/32) / (3 * 9/64) = 1 - 2/3 = 1/3.
    Catches: a wrong denominator (n-1 instead of n, N instead of N^2), |.| dropped, the 3 of the Binder line misplaced."""
    st = so.derived_stats([2, -2, 4, 0], 4)
    assert st["n"] == 4
    assert st["m"] == 0.25
    assert st["abs_m"] == 0.5
    assert st["m2"] == 0.375
    assert st["m4"] == 0.28125
    assert st["var_m"] == 0.3125
    assert abs(st["binder"] - 1.0 / 3.0) < 1e-15


def test_derived_stats_beyond_int64():
    """|M| = N = 2^30 (a fully ordered 32768^2 lattice): M^4 = 2^120 does not fit int64 (nor a double exactly when summed
    naively with smaller terms).  Three records (N, N, -N): <m> = 1/3, <|m|> = <m^2> = <m^4> = 1, Var = 1 - 1/9 = 8/9,
    U = 2/3.  Catches int64 / float accumulation of the power sums."""
    N = 2**30
    st = so.derived_stats(np.array([N, N, -N], dtype=np.int64), N)
    assert st["m"] == 1.0 / 3.0
    assert st["abs_m"] == 1.0 and st["m2"] == 1.0 and st["m4"] == 1.0
    assert abs(st["var_m"] - 8.0 / 9.0) < 1e-15
    assert abs(st["binder"] - 2.0 / 3.0) < 1e-15
    # one spin flipped in the second record: M = N - 2; exact rational values, far below double resolution of a float sum
    st = so.derived_stats([N, N - 2, -N], N)
    eps = 2.0 / N
    assert abs(st["abs_m"] - (1.0 - eps / 3.0)) < 1e-15
    assert abs(st["m2"] - (2.0 + (1.0 - eps) ** 2) / 3.0) < 1e-15
    assert abs(st["m4"] - (2.0 + (1.0 - eps) ** 4) / 3.0) < 1e-15


def test_binder_cumulant_special_values():
    """U = 1 - <m^4> / (3 <m^2>^2): constant |m| gives exactly 2/3 (ordered phase); a sample with one third of the weight
    at +-a and two thirds at 0 has <m^4> = 3 <m^2>^2, so U = 0 (the Gaussian value); all-zero records give NaN, not a
    division error.  Catches <m^2> and <m^4> exchanged, a missing square, a missing factor 3."""
    assert abs(so.derived_stats([5, -5, 5, 5, -5], 25)["binder"] - 2.0 / 3.0) < 1e-15
    st = so.derived_stats([6, -6, 0, 0, 0, 0], 36)
    assert st["binder"] == 0.0
    assert st["m"] == 0.0 and st["abs_m"] == 1.0 / 18.0
    assert abs(st["var_m"] - (72.0 / 6.0) / 36.0**2) < 1e-18 and st["var_m"] == st["m2"]
    assert math.isnan(so.derived_stats([0, 0, 0], 16)["binder"])


def test_energy_is_eq5_on_hand_made_configurations():
    """H(sigma, tau) = -sum_x [J sigma_x (tau_{x up} + tau_{x right}) + q sigma_x tau_x] (eq. 5).
    All +1 on an L x L torus: E_J = 2 L^2, E_q = L^2, H = -(2J + q) L^2.  One sigma spin flipped at x: the three bonds
    that touch it change sign: E_J = 2 L^2 - 4, E_q = L^2 - 2 (and C_x = C_y = L^2 - 4: two bonds each).  The bond sums come from the oracle's measure(), the
    expected integers from the counting argument.  Catches a sign error, J and q exchanged, a missing bond."""
    L = 6
    s = np.ones((L, L), dtype=np.int8)
    t = np.ones((L, L), dtype=np.int8)
    rec = so.measure(s, t)
    assert [int(v) for v in rec] == [36, 36, 72, 36, 36, 36]          # M_sigma, M_tau, E_J, E_q, C_x, C_y
    assert so.energy(0.7, 0.3, rec[2], rec[3]) == -(0.7 * 72 + 0.3 * 36)
    s[2, 3] = -1
    rec = so.measure(s, t)
    assert [int(v) for v in rec] == [34, 36, 68, 34, 32, 32]      # M_sigma, M_tau, E_J, E_q, C_x, C_y
    assert so.energy(1.0, 2.0, rec[2], rec[3]) == -(1.0 * 68 + 2.0 * 34)
    assert so.energy(0.5, 2.0, 10, -3) == -(0.5 * 10 + 2.0 * -3) == 1.0
    # which neighbours: sigma at x = (r, c) couples with tau at (r+1, c) [up], (r, c+1) [right], (r, c) [q] and nothing else.
    # sigma all +1 except x = (2, 3); tau all +1 except y = x + d.  With only tau_y flipped E_J = 68, E_q = 34; flipping
    # sigma_x as well changes the sign of its three bonds: a bond to tau_y goes from -1 back to +1, any other from +1 to -1.
    expected = {(0, 0): (64, 36), (1, 0): (68, 32), (0, 1): (68, 32), (-1, 0): (64, 32), (0, -1): (64, 32), (1, 1): (64, 32)}
    for (dr, dc), (EJ, Eq) in expected.items():
        t = np.ones((L, L), dtype=np.int8)
        t[(2 + dr) % L, (3 + dc) % L] = -1
        rec = so.measure(np.ones((L, L), dtype=np.int8), t)
        assert (int(rec[2]), int(rec[3])) == (68, 34), (dr, dc)
        rec = so.measure(s, t)
        assert (int(rec[2]), int(rec[3])) == (EJ, Eq), (dr, dc)
