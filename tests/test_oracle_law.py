"""The oracle against what the paper and the mathematics fix: closed forms, the exact 3x3 transition
matrix, the stationary measure the paper states, invariants.  CPU only; citations are PAPER.md lines."""
import math

import numpy as np
import pytest

from oracle import shaken_oracle as so
from tests import pins

needs_curand = pytest.mark.skipif(not pins.curand_available(), reason="libcurand not found")


def chi2_ok(counts, probs, n, z=5.0):
    """Pearson chi^2 against exact cell probabilities; cells with tiny expectation are pooled.
    Accept if chi^2 < dof + z*sqrt(2 dof)."""
    exp = probs * n
    big = exp >= 5
    c = np.append(counts[big], counts[~big].sum())
    e = np.append(exp[big], exp[~big].sum())
    keep = e > 0
    chi2 = ((c[keep] - e[keep]) ** 2 / e[keep]).sum()
    dof = keep.sum() - 1
    return chi2 < dof + z * math.sqrt(2 * dof), chi2, dof


# ----------------------------------------------------------------------------- J = q = 0
@needs_curand
def test_zero_couplings_spin_is_top_bit_of_the_random_word():
    """J=q=0: every field is 0, P(+)=1/2, so the new spin is +1 iff the word's top bit is 0 -- whatever the
    neighbours are.  Words from cuRAND.  Catches a threshold off by a factor 2 or a mis-indexed word."""
    L, seed = 8, 31
    o = so.Oracle(L, 2, seed)
    o.init(0)
    o.run(0.0, 0.0, 2, 0)
    for ch in range(2):
        w_tau = pins.curand_site_words(seed, ch, 2, L * L)     # t=1, half 0
        w_sig = pins.curand_site_words(seed, ch, 3, L * L)     # t=1, half 1
        assert np.array_equal(o.get_spins(1)[ch].reshape(-1), np.where(w_tau < 2**31, 1, -1))
        assert np.array_equal(o.get_spins(0)[ch].reshape(-1), np.where(w_sig < 2**31, 1, -1))


def test_zero_couplings_magnetisation_is_binomial():
    o = so.Oracle(32, 64, 5)
    o.init(1)
    o.run(0.0, 0.0, 3, 1)
    M = o.observables()[:, :, 0].astype(np.float64)              # 2 Bin(1024, 1/2) - 1024: mean 0, var 1024
    z = M.mean() / math.sqrt(1024 / M.size)
    assert abs(z) < 5
    assert abs(M.var() / 1024 - 1) < 0.25


# ----------------------------------------------------------------------------- J = 0: closed-form contraction
def test_J0_magnetisation_contracts_by_tanh_q_per_half_step():
    """J=0: sites decouple, sigma_x -> tau_x -> sigma'_x is a two-state chain with E[new|old] = tanh(q) old
    when P(+|h) = (1+tanh h)/2.  From all +1: E M_tau(k)/N = rho^(2k-1), E M_sigma(k)/N = rho^(2k).
    Catches the other heat-bath normalisations (tanh 2q, e^{-h}) and a half-step applied twice or skipped."""
    q, L, n_chains, n_steps = 0.4, 16, 400, 4
    rho = math.tanh(q)
    o = so.Oracle(L, n_chains, 17)
    o.init(1)
    o.run(0.0, q, n_steps, 1)
    rec = o.observables().astype(np.float64)
    N = L * L
    for k in range(1, n_steps + 1):
        for col, power in ((0, 2 * k), (1, 2 * k - 1)):
            mean = rec[k - 1, :, col].mean() / N
            var_site = 1 - rho ** (2 * power)
            se = math.sqrt(var_site / (N * n_chains))
            assert abs(mean - rho**power) < 5 * se, (k, col, mean, rho**power)
    # and from all -1 the sign flips
    o.init(-1)
    o.run(0.0, q, 1, 1)
    mean = o.observables()[0, :, 0].mean() / N
    assert abs(mean + rho**2) < 5 * math.sqrt(1.0 / (N * n_chains))
    # E_q = sum sigma'_x tau_x has mean rho per site at any time >= 1 (one q-bond in equilibrium with its field)
    eq = rec[:, :, 3].mean() / N
    assert abs(eq - rho) < 5 * math.sqrt(1.0 / (N * n_chains * n_steps))


# ----------------------------------------------------------------------------- 3x3 torus, exact
J3, Q3 = 0.4, 0.3


def test_exact_3x3_kernels_satisfy_what_the_paper_states():
    """Pins the test's own matrices to the paper before they judge the oracle: rows sum to 1; eq. (15)'s product
    form equals e^{-H}/Z_sigma; pi_s = Z_sigma/Z (:180-186) is stationary for P = P15 P16 and satisfies detailed
    balance; pi_2 (eq. 6 :98) is invariant under each half-step."""
    P15, P16, Zs = pins.exact_kernels_3x3(J3, Q3)
    assert np.allclose(P15.sum(1), 1, atol=1e-13) and np.allclose(P16.sum(1), 1, atol=1e-13)
    cfgs = pins.all_configs(3)
    # eq. (15): P((s,t),(s,t')) = e^{-H(s,t')}/Z_s  -- check on a sample of pairs
    rng = np.random.default_rng(0)
    for a, b in rng.integers(0, 512, size=(40, 2)):
        w = math.exp(-pins.hamiltonian_pair(cfgs[a], cfgs[b], J3, Q3))
        assert abs(P15[a, b] - w / Zs[a]) < 1e-13
    # eq. (16): P((s,t),(s',t)) = e^{-H(s',t)}/Z_t with Z_t = sum_eta e^{-H(eta,t)}: full check through the weight matrix
    Wm = np.exp(-np.array([[pins.hamiltonian_pair(cfgs[a], cfgs[b], J3, Q3) for b in range(512)] for a in range(512)]))
    assert np.allclose(Wm.sum(1), Zs, rtol=1e-12)                         # Z_sigma = sum_tau e^{-H}
    Zt = Wm.sum(0)
    assert np.allclose(P16, (Wm / Zt[None, :]).T, atol=1e-13)           # P16[t, s'] = W[s', t]/Z_t
    P = P15 @ P16                                                         # shaken kernel P^square (:178)
    pi_s = Zs / Zs.sum()
    assert np.allclose(pi_s @ P, pi_s, atol=1e-14)
    flow = pi_s[:, None] * P
    assert np.allclose(flow, flow.T, atol=1e-15)                          # detailed balance (reading 13)
    pi2 = Wm / Wm.sum()                                                   # eq. (6)
    assert np.allclose((pi2.sum(1)[:, None] * P15), pi2, atol=1e-15)      # half-step 0 resamples tau | sigma
    assert np.allclose(pi2.sum(1), pi_s, atol=1e-15)                      # sigma-marginal of pi_2 is pi_s (:198)


@pytest.mark.parametrize("sigma0_id", [0b000010110, 0b111111111, 0b100000001])
def test_oracle_one_and_two_step_law_on_3x3_matches_exact_matrix(sigma0_id):
    """Empirical law of sigma after 1 and 2 full steps from a fixed sigma_0, over 400k independent chains,
    against rows of P and P^2 built from eq. (15)-(16) (chi^2).  Also the law of tau after the first half-step
    against eq. (15) alone.  Catches: both halves using the same direction, halves swapped, transposed
    neighbour roles -- the start configurations are not reflection symmetric."""
    n = 400_000
    T = so.thresholds(J3, Q3)
    P15, P16, _ = pins.exact_kernels_3x3(J3, Q3, table=T)
    P = P15 @ P16
    s0 = pins.all_configs(3)[sigma0_id]
    o = so.Oracle(3, n, 2024)
    o.set_spins(0, np.broadcast_to(s0, (n, 3, 3)).copy())
    o.run(J3, Q3, 1, 0)
    tau_ids = pins.config_id(o.get_spins(1))
    sig_ids = pins.config_id(o.get_spins(0))
    ok, chi2, dof = chi2_ok(np.bincount(tau_ids, minlength=512), P15[sigma0_id], n)
    assert ok, ("tau | sigma0", chi2, dof)
    ok, chi2, dof = chi2_ok(np.bincount(sig_ids, minlength=512), P[sigma0_id], n)
    assert ok, ("sigma1 | sigma0", chi2, dof)
    o.run(J3, Q3, 1, 0)
    ok, chi2, dof = chi2_ok(np.bincount(pins.config_id(o.get_spins(0)), minlength=512), (P @ P)[sigma0_id], n)
    assert ok, ("sigma2 | sigma0", chi2, dof)
    # a wrong reading must FAIL the same test (power check): swap the halves' directions
    Pw = P16 @ P15
    bad, _, _ = chi2_ok(np.bincount(sig_ids, minlength=512), Pw[sigma0_id], n)
    if sigma0_id not in (0b111111111,):
        assert not bad


def test_oracle_long_run_occupancy_matches_stationary_measure_on_3x3():
    """After 60 steps from an iid start the law of sigma is pi_s = Z_sigma/Z up to mixing error
    (second eigenvalue^60 is negligible here)."""
    n = 300_000
    T = so.thresholds(J3, Q3)
    P15, P16, _ = pins.exact_kernels_3x3(J3, Q3, table=T)
    P = P15 @ P16
    ev = np.sort(np.abs(np.linalg.eigvals(P)))[::-1]
    assert ev[1] ** 60 < 1e-6
    w, v = np.linalg.eig(P.T)
    pi = np.real(v[:, np.argmax(np.real(w))])
    pi = pi / pi.sum()
    _, _, Zs = pins.exact_kernels_3x3(J3, Q3)
    assert np.allclose(pi, Zs / Zs.sum(), atol=1e-8)                      # quantised table vs exact pi_s
    o = so.Oracle(3, n, 77)
    o.init(0)
    o.run(J3, Q3, 60, 0)
    ok, chi2, dof = chi2_ok(np.bincount(pins.config_id(o.get_spins(0)), minlength=512), pi, n)
    assert ok, (chi2, dof)


# ----------------------------------------------------------------------------- invariants
def test_two_forms_of_the_hamiltonian_agree():
    """eq. (5): sum_x s_x (t_up + t_right) = sum_x t_x (s_down + s_left)."""
    rng = np.random.default_rng(3)
    for L in (3, 4, 7, 16):
        s = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
        t = rng.choice(np.array([-1, 1], dtype=np.int8), size=(L, L))
        m = so.measure(s, t)
        assert np.array_equal(m, pins.brute_observables(s, t))
        s64, t64 = s.astype(np.int64), t.astype(np.int64)
        second_form = (t64 * (np.roll(s64, 1, axis=0) + np.roll(s64, 1, axis=1))).sum()
        assert m[2] == second_form
        assert (m[0] - L * L) % 2 == 0
    ones = np.ones((8, 8), dtype=np.int8)
    assert list(so.measure(ones, ones)) == [64, 64, 128, 64, 64, 64]
    assert list(so.measure(ones, -ones)) == [64, -64, -128, -64, 64, 64]


def test_run_is_resumable_and_chains_are_independent_of_batch_size():
    """Counter-based randomness: run(a); run(b) == run(a+b); chain c does not depend on how many chains exist;
    set_step replays a step."""
    J, q = 0.5, 0.7
    a = so.Oracle(12, 3, 9); a.init(0); a.run(J, q, 7, 1)
    b = so.Oracle(12, 3, 9); b.init(0); b.run(J, q, 3, 1); b.run(J, q, 4, 1)
    assert np.array_equal(a.get_spins(0), b.get_spins(0)) and np.array_equal(a.get_spins(1), b.get_spins(1))
    assert np.array_equal(a.observables(), b.observables())
    c = so.Oracle(12, 5, 9); c.init(0); c.run(J, q, 7, 1)
    assert np.array_equal(c.get_spins(0)[:3], a.get_spins(0))
    assert np.array_equal(c.observables()[:, :3], a.observables())
    d = so.Oracle(12, 3, 10); d.init(0); d.run(J, q, 7, 0)
    assert not np.array_equal(d.get_spins(0), a.get_spins(0))
    e = so.Oracle(12, 3, 9 + 2**32); e.init(0)
    assert not np.array_equal(e.get_spins(0), so.Oracle(12, 3, 9).get_spins(0))
    # replay of step 5 from a snapshot
    f = so.Oracle(12, 3, 9); f.init(0); f.run(J, q, 5, 0)
    snap_s, snap_t = f.get_spins(0), f.get_spins(1)
    f.run(J, q, 1, 0)
    g = so.Oracle(12, 3, 9); g.set_spins(0, snap_s); g.set_spins(1, snap_t); g.step = 5; g.run(J, q, 1, 0)
    assert np.array_equal(f.get_spins(0), g.get_spins(0))
    # obs_every counts global 1-based steps
    h = so.Oracle(12, 1, 9); h.init(0); h.run(J, q, 4, 3); h.run(J, q, 5, 3)
    assert h.observables().shape[0] == 3
    # grid form with equal couplings == scalar form
    k = so.Oracle(12, 3, 9); k.init(0); k.run_grid([J] * 3, [q] * 3, 7, 1)
    assert np.array_equal(k.observables(), a.observables())


def test_monotone_coupling_and_coalescence():
    """the dynamics preserves the partial order under shared randomness (J, q >= 0); top and bottom
    chains coalesce at weak coupling."""
    L, J, q = 10, 0.3, 0.4
    rng = np.random.default_rng(8)
    lo = rng.choice(np.array([-1, 1], dtype=np.int8), size=(1, L, L))
    hi = np.maximum(lo, rng.choice(np.array([-1, 1], dtype=np.int8), size=(1, L, L)))
    a = so.Oracle(L, 1, 4); a.set_spins(0, lo)
    b = so.Oracle(L, 1, 4); b.set_spins(0, hi)
    top = so.Oracle(L, 1, 4); top.init(1)
    bot = so.Oracle(L, 1, 4); bot.init(-1)
    coalesced = None
    for t in range(200):
        for o in (a, b, top, bot):
            o.run(J, q, 1, 0)
        assert np.all(a.get_spins(0) <= b.get_spins(0)) and np.all(a.get_spins(1) <= b.get_spins(1))
        assert np.all(bot.get_spins(0) <= a.get_spins(0)) and np.all(b.get_spins(0) <= top.get_spins(0))
        if coalesced is None and np.array_equal(top.get_spins(0), bot.get_spins(0)):
            coalesced = t
    assert coalesced is not None and coalesced < 150
    assert np.array_equal(a.get_spins(0), top.get_spins(0))


def test_global_spin_flip_symmetry_with_complemented_words():
    """T(h)+T(-h)=2^32 => flipping sigma_0 and replacing every word r by 2^32-1-r flips the whole trajectory."""
    L, J, q = 9, 0.6, 0.35
    a = so.Oracle(L, 2, 12); a.init(0)
    b = so.Oracle(L, 2, 12); b.set_spins(0, -a.get_spins(0)); b.set_spins(1, -a.get_spins(1)); b.set_complement(True)
    a.run(J, q, 5, 1); b.run(J, q, 5, 1)
    assert np.array_equal(a.get_spins(0), -b.get_spins(0)) and np.array_equal(a.get_spins(1), -b.get_spins(1))
    ra, rb = a.observables(), b.observables()
    assert np.array_equal(ra[:, :, :2], -rb[:, :, :2]) and np.array_equal(ra[:, :, 2:], rb[:, :, 2:])


def test_saturated_limits_fix_the_neighbour_conventions():
    """J=0, q=20: T saturates, half 0 copies sigma into tau and half 1 copies it back.
    q=0, J=20: tau'_y is forced where sigma_down and sigma_left agree; e.g. sigma=+1 only at (r,c)=(0,1) and (1,0)
    forces tau'_(1,1)=+1; mirrored with up/right for half 1."""
    L = 6
    rng = np.random.default_rng(1)
    s0 = rng.choice(np.array([-1, 1], dtype=np.int8), size=(1, L, L))
    o = so.Oracle(L, 1, 3); o.set_spins(0, s0); o.run(0.0, 20.0, 1, 0)
    assert np.array_equal(o.get_spins(1), s0) and np.array_equal(o.get_spins(0), s0)
    # forced sites with q = 0
    s = -np.ones((1, L, L), dtype=np.int8)
    s[0, 0, 1] = 1   # (r=0, c=1): the down neighbour of (1,1)
    s[0, 1, 0] = 1   # (r=1, c=0): the left neighbour of (1,1)
    for seed in range(20):
        o = so.Oracle(L, 1, seed); o.set_spins(0, s)
        # run only half 0 by inspecting tau after one step: tau is written by half 0 and not touched by half 1
        o.run(20.0, 0.0, 1, 0)
        tau = o.get_spins(1)[0]
        assert tau[1, 1] == 1
        # sites whose down and left neighbours are both -1 are forced to -1
        down = np.roll(s[0], 1, axis=0); left = np.roll(s[0], 1, axis=1)
        assert np.all(tau[(down == -1) & (left == -1)] == -1)
        # half 1: sigma'_x forced by tau_up, tau_right
        sig = o.get_spins(0)[0]
        up = np.roll(tau, -1, axis=0); right = np.roll(tau, -1, axis=1)
        assert np.all(sig[(up == 1) & (right == 1)] == 1) and np.all(sig[(up == -1) & (right == -1)] == -1)


def test_q0_decouples_into_rings_with_textbook_1d_correlations():
    """q=0: the honeycomb falls apart into rings of 2L spins running NW-SE:
    sigma_(r,c) - tau_(r,c+1) ... ; equilibrium <s_0 s_k> on a ring of n=2L spins with coupling J is
    (u^k + u^(n-k))/(1+u^n), u = tanh J.  tau_y is bonded to sigma_down(y) and sigma_left(y) (eq. 5), so the ring
    through sigma_(r,c) is sigma_(r,c) - tau_(r+1,c) - sigma_(r+1,c-1) - tau_(r+2,c-1) - ...; sites on different
    rings are uncorrelated."""
    L, J, n_chains = 6, 0.5, 6000
    u = math.tanh(J)
    n = 2 * L
    o = so.Oracle(L, n_chains, 123); o.init(0); o.run(J, 0.0, 40, 0)
    s = o.get_spins(0).astype(np.float64)
    t = o.get_spins(1).astype(np.float64)
    se = 1 / math.sqrt(n_chains * L * L)
    # J-bond: sigma_x with tau_up(x) and tau_right(x): one bond apart
    c1 = (u + u ** (n - 1)) / (1 + u**n)
    assert abs((s * np.roll(t, -1, axis=1)).mean() - c1) < 6 * se
    assert abs((s * np.roll(t, -1, axis=2)).mean() - c1) < 6 * se
    # y=(r+1,c): sigma_(r,c) = sigma_down(y) and sigma_(r+1,c-1) = sigma_left(y): two bonds apart
    c2 = (u**2 + u ** (n - 2)) / (1 + u**n)
    nwse = (s * np.roll(np.roll(s, -1, axis=1), 1, axis=2)).mean()     # s_(r,c) s_(r+1,c-1)
    assert abs(nwse - c2) < 6 * se
    # the other diagonal (r+1, c+1) lies on a different ring: uncorrelated
    swne = (s * np.roll(np.roll(s, -1, axis=1), -1, axis=2)).mean()
    assert abs(swne) < 6 * se
    # sigma_(r,c) lies on ring (r+c) mod L, tau_(r,c) on ring (r+c-1): no bond at q=0, uncorrelated
    assert abs((s * t).mean()) < 6 * se
