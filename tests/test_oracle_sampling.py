"""Pin for the oracle's Propp-Wilson driver: on the 3 x 3 torus the samples must follow the
stationary measure of the two-half-step kernel, which is built exactly (512 x 512) from eq. (15)-(16) with the
oracle-independent helper of tests/pins.py.  An exact sampler has NO burn-in bias, so a plain chi-square applies.
CPU only."""
import math

import numpy as np

from oracle import shaken_oracle as so
from tests import pins


def test_propp_wilson_samples_follow_the_exact_stationary_measure_on_3x3():
    J, q, n_pairs, seed = 0.35, 0.5, 6000, 2024
    table = so.thresholds(J, q)
    P15, P16, _ = pins.exact_kernels_3x3(J, q, table=table)      # the quantised law the integer compare realises
    P = P15 @ P16
    w, v = np.linalg.eig(P.T)
    pi = np.real(v[:, np.argmin(np.abs(w - 1.0))])
    pi = pi / pi.sum()
    assert np.all(pi > 0) and np.allclose(pi @ P, pi, atol=1e-13)

    o = so.Oracle(3, 2 * n_pairs, seed)
    o.set_coupling(2)
    samples, T = so.propp_wilson(o, np.full(2 * n_pairs, J), np.full(2 * n_pairs, q))
    assert samples.shape == (n_pairs, 3, 3) and T >= 1 and (T & (T - 1)) == 0
    # state index in the enumeration of pins.all_configs
    cfgs = pins.all_configs(3)
    key = {c.astype(np.int8).tobytes(): i for i, c in enumerate(cfgs)}
    idx = np.array([key[s.tobytes()] for s in samples])
    counts = np.bincount(idx, minlength=512).astype(np.float64)
    expected = n_pairs * pi
    big = expected >= 5.0                                          # pool the rare states into one bin
    chi2 = ((counts[big] - expected[big]) ** 2 / expected[big]).sum()
    rest_e, rest_o = expected[~big].sum(), counts[~big].sum()
    dof = int(big.sum()) - 1
    if rest_e >= 5.0:
        chi2 += (rest_o - rest_e) ** 2 / rest_e
        dof += 1
    assert chi2 < dof + 5.0 * math.sqrt(2.0 * dof), (chi2, dof)
    # the same random numbers give the same draw: a second call with the same base reproduces it, another base does not
    again, T2 = so.propp_wilson(o, np.full(2 * n_pairs, J), np.full(2 * n_pairs, q))
    assert T2 == T and np.array_equal(again, samples)
    other, _ = so.propp_wilson(o, np.full(2 * n_pairs, J), np.full(2 * n_pairs, q), base=(1 << 40) + (1 << 20))
    assert not np.array_equal(other, samples)
