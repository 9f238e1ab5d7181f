"""Pins of the oracle against things other than itself (CPU only).

Each test names the mistake it would catch.  Citations are PAPER.md lines.
"""
import math
import os

import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import workloads
from tests import pins

needs_curand = pytest.mark.skipif(not pins.curand_available(), reason="libcurand not found")


# ----------------------------------------------------------------------------- Philox4x32-10
@needs_curand
def test_philox_matches_curand_host_generator():
    """Library-routine pin: cuRAND's host Philox4_32_10 generator.  Catches a wrong multiplier, a wrong
    Weyl constant, swapped hi/lo words, a wrong round count or key schedule."""
    rng = np.random.default_rng(1234)
    for seed in [0, 1, 0xDEADBEEF, 0x123456789ABCDEF0, 2**64 - 1]:
        key = (seed & 0xFFFFFFFF, seed >> 32)
        for k in [0, 1, 2**32 - 1, 2**32, int(rng.integers(0, 2**45))]:
            grp = pins.curand_host_stream(seed, k, 300)
            for g in [0, 1, 2, 17, 255, 299]:
                ctr = (k & 0xFFFFFFFF, (k >> 32) & 0xFFFFFFFF, g, 0)
                assert np.array_equal(so.philox4x32_10(ctr, key), grp[g]), (seed, k, g)


def test_philox_counter_word3_and_bijection_sanity():
    """Word 3 of the counter is not reachable through the host generator (pinned on the GPU against
    curand_Philox4x32_10 in tests/test_gpu_philox.py); here: it must matter, and distinct counters must
    give distinct blocks (Philox is a bijection of the counter for a fixed key)."""
    key = (7, 9)
    seen = set()
    for c3 in range(64):
        for c0 in range(8):
            out = tuple(int(v) for v in so.philox4x32_10((c0, 1, 2, c3), key))
            assert out not in seen
            seen.add(out)
    # bit balance of 4*20000 words: each bit set about half the time
    ws = np.concatenate([so.philox4x32_10((i, 0, 0, 0xFFFFFFFF), key) for i in range(20000)])
    ones = np.array([(ws >> b & 1).mean() for b in range(32)])
    assert np.all(np.abs(ones - 0.5) < 5 * 0.5 / math.sqrt(ws.size))


# ----------------------------------------------------------------------------- critical curve (golden, helper)
def test_critical_curve_values_printed_by_the_paper():
    path = os.path.join(os.path.dirname(__file__), "golden", "critical_curve.txt")
    vals = {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        label, value, digits = line.split()[:3]
        vals[label] = (float(value), int(digits))
    v, d = vals["square_limit"]
    assert abs(workloads.critical_J(50.0) - v) < 10**-d                # eq. (13) :147 (the paper truncates: one unit of the last digit)
    assert abs(math.atanh(math.sqrt(2) - 1) - v) < 10**-d
    v, d = vals["honeycomb_fix"]
    # J_c(q) = q has the root tanh^2 J = 1/3  (eq. 11 with J=q) -> atanh(1/sqrt 3)
    root = math.atanh(1 / math.sqrt(3))
    assert abs(root - v) < 10**-d                                   # :151
    assert abs(workloads.critical_J(root) - root) < 1e-12
    # eq. (11): 1 = 2 tanh J tanh q + tanh^2 J along the curve
    for q in [0.05, 0.3, 1.0, 2.5]:
        J = workloads.critical_J(q)
        assert abs(2 * math.tanh(J) * math.tanh(q) + math.tanh(J) ** 2 - 1) < 1e-12


# ----------------------------------------------------------------------------- thresholds
CFG_COUPLINGS = [(0.5, 0.5), (0.6585, 0.6585), (0.7, 0.7), (0.45, 10.0), (0.44, 0.66), (0.05, 0.1),
                 (1.2, 20.0), (0.05 + 7 * (1.15 / 15.0), 5.0), (0.99, 0.5), (2.0, 0.03), (0.0, 0.0),
                 (0.0, 1.0), (1.0, 0.0), (-0.3, 0.4), (0.3, -0.4)]


def test_threshold_table_against_exact_decimal_arithmetic():
    """Closed form: T = round(2^32 e^h / (2 cosh h)).  Catches a wrong sign of h, a factor 2 in
    the exponent (tanh h vs tanh 2h), wrong (k, c) -> field map, wrong index order."""
    for J, q in CFG_COUPLINGS:
        T = so.thresholds(J, q)
        for k in range(3):
            for c in range(2):
                h = pins.field(J, q, k, c)
                real = pins.exact_threshold_real(h)
                got = int(T[2 * k + c])
                assert 1 <= got <= 2**32 - 1
                clamped = min(max(real, 1), 2**32 - 1)
                # double evaluation: relative error of p a few ulp -> a few 1e-7 absolute on the 2^32 scale
                assert abs(got - float(clamped)) <= 0.5 + 4e-6, (J, q, k, c, got, real)
        # the exact table agrees entry by entry unless the real value sits within 4e-6 of a half-integer
        ex = pins.exact_table(J, q)
        for i in range(6):
            if abs(float(ex[i]) - float(T[i])) != 0:
                frac = float(pins.exact_threshold_real(pins.field(J, q, i // 2, i % 2)) % 1)
                assert abs(frac - 0.5) < 4e-6


def test_threshold_symmetry_monotone_saturation():
    assert so.threshold(0.0) == 2**31
    hs = np.linspace(-30, 30, 2001)
    T = np.array([so.threshold(float(h)) for h in hs], dtype=np.int64)
    assert np.all(np.diff(T) >= 0)                        # monotone in the field
    assert np.all(T + T[::-1] == 2**32)                   # P(+|h) + P(+|-h) = 1 exactly (spin-flip symmetry)
    assert T[0] == 1 and T[-1] == 2**32 - 1               # both outcomes keep non-zero probability (eq. 15-16)
    # tanh form: P(+) = (1 + tanh h)/2
    for h in [0.1, 0.7, 2.1, -1.3]:
        assert abs(so.threshold(h) / 2**32 - 0.5 * (1 + math.tanh(h))) < 2**-31
    # saturation values quoted in DESIGN.md (cfg 5: q=10, J=0.45)
    assert so.threshold(10.0) == 2**32 - 9
    assert so.threshold(10.9) == 2**32 - 1


# ----------------------------------------------------------------------------- half-steps vs brute force with cuRAND words
@needs_curand
@pytest.mark.parametrize("L,J,q,seed,chain", [(8, 0.5, 0.5, 1, 0), (6, 0.3, 1.1, 99, 2), (3, 0.8, 0.2, 5, 1), (5, 0.44, 0.66, 2**40 + 3, 0)])
def test_full_steps_against_numpy_brute_force_with_curand_words(L, J, q, seed, chain):
    """Brute force on tiny tori: eq. (15)-(16) with numpy roll, exact decimal thresholds and random words from
    cuRAND (NOT the oracle's Philox).  Catches: wrong neighbour direction in either half, wrong half order,
    wrong counter layout (site>>2, chain, g), wrong word (site&3), <= instead of <, in-place hazards."""
    n_chains = chain + 1
    o = so.Oracle(L, n_chains, seed)
    rng = np.random.default_rng(seed % 1000)
    s0 = rng.choice(np.array([-1, 1], dtype=np.int8), size=(n_chains, L, L))
    t0 = rng.choice(np.array([-1, 1], dtype=np.int8), size=(n_chains, L, L))
    o.set_spins(0, s0)
    o.set_spins(1, t0)
    table = pins.exact_table(J, q)
    assert np.array_equal(table, so.thresholds(J, q).astype(np.uint64))
    sigma = s0[chain].copy()
    n_steps = 3
    o.run(J, q, n_steps, 1)
    rec = o.observables()
    assert rec.shape == (n_steps, n_chains, 6)
    # replay
    o2 = so.Oracle(L, n_chains, seed)
    o2.set_spins(0, s0)
    o2.set_spins(1, t0)
    for t in range(n_steps):
        tau = pins.brute_half_step(sigma, 0, table, pins.curand_site_words(seed, chain, 2 * t, L * L))
        sigma = pins.brute_half_step(tau, 1, table, pins.curand_site_words(seed, chain, 2 * t + 1, L * L))
        o2.run(J, q, 1, 0)
        assert np.array_equal(o2.get_spins(1)[chain], tau), t
        assert np.array_equal(o2.get_spins(0)[chain], sigma), t
        assert np.array_equal(rec[t, chain], pins.brute_observables(sigma, tau)), t
    assert o2.step == n_steps


@needs_curand
def test_iid_init_against_curand_words():
    """Init stream: counter (site>>2, chain, which, 0xFFFFFFFF) is out of the host generator's reach (word 3),
    so here only the law is pinned: +1 iff word < 2^31, fair, sigma and tau differ, chains differ."""
    o = so.Oracle(64, 3, 1)
    o.init(0)
    s, t = o.get_spins(0), o.get_spins(1)
    assert set(np.unique(s)) == {-1, 1}
    for a in (s, t):
        for ch in range(3):
            m = a[ch].astype(np.int64).sum()
            assert abs(m) < 5 * 64                          # 5 sigma of 2 Bin(4096, 1/2) - 4096
    assert not np.array_equal(s, t) and not np.array_equal(s[0], s[1])
    # direct recomputation from the pinned Philox function
    key = (1, 0)
    for which, arr in ((0, s), (1, t)):
        for ch in range(3):
            for call in [0, 1, 500, 1023]:
                w = so.philox4x32_10((call, ch, which, 0xFFFFFFFF), key)
                exp = np.where(w < 2**31, 1, -1)
                assert np.array_equal(arr[ch].reshape(-1)[4 * call: 4 * call + 4], exp)


@needs_curand
def test_row_restricted_half_step_against_numpy_brute_force_with_curand_words():
    """oracle.half_step_rows (used for full-size spot checks on the GPU box) is the same per-site statement
    restricted to a band of rows: pinned on a small torus against eq. (15)/(16) with numpy roll, exact decimal
    thresholds and cuRAND's words; also equal to the context's full half-steps."""
    L, seed, chain, J, q, t = 12, 77, 3, 0.45, 0.9, 5
    rng = np.random.default_rng(3)
    src = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
    table = pins.exact_table(J, q)
    for half in (0, 1):
        full = pins.brute_half_step(src, half, table, pins.curand_site_words(seed, chain, 2 * t + half, L * L))
        for r0, nrows in [(0, L), (0, 1), (L - 1, 1), (4, 5)]:
            got = so.half_step_rows(src, seed, chain, J, q, t, half, r0, nrows)
            assert np.array_equal(got, full[r0:r0 + nrows]), (half, r0, nrows)
    # and the context path: one full step from (src, anything) = half 0 then half 1
    o = so.Oracle(L, chain + 1, seed)
    s0 = np.ones((chain + 1, L, L), dtype=np.int8)
    s0[chain] = src
    o.set_spins(0, s0)
    o.step = t
    o.run(J, q, 1, 0)
    tau = so.half_step_rows(src, seed, chain, J, q, t, 0, 0, L)
    assert np.array_equal(o.get_spins(1)[chain], tau)
    assert np.array_equal(o.get_spins(0)[chain], so.half_step_rows(tau, seed, chain, J, q, t, 1, 0, L))
