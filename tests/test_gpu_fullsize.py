"""Full-size parity (``-m gpu``): BASELINE.json configs 2-5 at their real L and chain count, in the launch
configuration bench.py times.  The oracle is too slow for full-length runs here (SURVEY 8(c) last row), so:

* complete lattices are compared for the first steps, and
* *snapshot induction*: the GPU state after k steps is downloaded, the oracle advances ONE step from it with
  ``step = k`` (legal because the randomness is indexed by the step), and the result must equal the GPU state
  after k+1 steps, spins and records;
* at L = 32768 (cfg 5, 2.1e9 site updates per step) the oracle computes sampled bands of rows of each half-step
  (``oracle.half_step_rows``) from the downloaded source layer, and the six sums by brute force;
* whole-lattice steps at L = 32768 (packed) and L = 65536 (int8), and the FULL-LENGTH cfg 2 run (10^4 steps), use the same
  row function over ALL rows, the bands spread over the host cores (tests/rowsplit.py).
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import shaken, workloads
from tests import rowsplit

pytestmark = pytest.mark.gpu


def host_memory_gb() -> float:
    try:
        import psutil

        return psutil.virtual_memory().available / 2**30
    except Exception:
        return 0.0


def oracle_step_from(s: shaken.Shaken, w, J, q, n_steps=1, obs_every=1):
    o = so.Oracle(w.L, w.n_chains, w.seed)
    o.set_spins(0, s.get_spins(0))
    o.set_spins(1, s.get_spins(1))
    o.step = s.step
    o.run_grid(np.asarray(J), np.asarray(q), n_steps, obs_every)
    return o


def test_cfg2_first_steps_and_snapshot_induction():
    w = workloads.config(2)                       # L=1024, J=q=0.6585, all +1, seed 7, obs every 10
    o = so.Oracle(w.L, 1, w.seed)
    o.init(w.init)
    o.run(w.J[0], w.q[0], 20, w.obs_every)
    with shaken.Shaken(w.L, 1, w.seed, max_records=64) as s:
        s.init(w.init)
        s.run(w.J[0], w.q[0], 20, w.obs_every)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.get_spins(1), o.get_spins(1))
        assert np.array_equal(s.observables(), o.observables()) and s.num_records == 2
        s.run(w.J[0], w.q[0], 389, w.obs_every)   # to step 409: next step is recorded
        o2 = oracle_step_from(s, w, w.J, w.q, 1, w.obs_every)
        n0 = s.num_records
        s.run(w.J[0], w.q[0], 1, w.obs_every)
        assert s.step == 410 and s.num_records == n0 + 1
        assert np.array_equal(s.get_spins(0), o2.get_spins(0)) and np.array_equal(s.get_spins(1), o2.get_spins(1))
        assert np.array_equal(s.observables()[-1], o2.observables()[-1])


def test_cfg3_grid_512_chains_first_step_and_snapshot_induction():
    w = workloads.config(3)                       # 512 chains x 512^2, iid start, seed 11, obs every step
    J, q = w.J_array(), w.q_array()
    with shaken.Shaken(w.L, w.n_chains, w.seed, max_records=32) as s:
        s.init(w.init)
        o = so.Oracle(w.L, w.n_chains, w.seed)
        o.init(w.init)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.get_spins(1), o.get_spins(1))
        o.run_grid(J, q, 1, 1)
        s.run_grid(J, q, 1, 1)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.get_spins(1), o.get_spins(1))
        assert np.array_equal(s.observables(), o.observables())
        del o
        s.run_grid(J, q, 24, 1)
        o2 = oracle_step_from(s, w, J, q, 1, 1)
        s.run_grid(J, q, 1, 1)
        assert s.step == 26
        assert np.array_equal(s.get_spins(0), o2.get_spins(0)) and np.array_equal(s.get_spins(1), o2.get_spins(1))
        assert np.array_equal(s.observables()[-1], o2.observables()[-1])
        # frozen rows of the grid (q = 20): sigma and tau stay locked together, E_q = L^2 from the first record on
        rec = s.observables()
        assert np.all(rec[:, 448:, 3] == w.L * w.L)


def test_cfg4_headline_lattice_snapshot_induction():
    w = workloads.config(4)                       # L=16384, J=q=0.7, all +1, seed 3, all six sums every step
    with shaken.Shaken(w.L, 1, w.seed, max_records=8) as s:
        s.init(w.init)
        s.run(w.J[0], w.q[0], 3, 1)
        o = oracle_step_from(s, w, w.J, w.q, 1, 1)
        rec3 = s.observables()[-1, 0].copy()
        sg, ta = s.get_spins(0), s.get_spins(1)
        assert np.array_equal(rec3, so.measure(sg[0], ta[0]))          # records of step 3 by brute force
        del sg, ta
        s.run(w.J[0], w.q[0], 1, 1)
        assert s.step == 4 and s.num_records == 4
        assert np.array_equal(s.get_spins(1), o.get_spins(1)), "tau after step 4"
        assert np.array_equal(s.get_spins(0), o.get_spins(0)), "sigma after step 4"
        assert np.array_equal(s.observables()[-1], o.observables()[-1])


def test_cfg5_packed_32768_sampled_rows_and_brute_force_sums():
    w = workloads.config(5)                       # L=32768 packed, q=10, J=0.45, iid, seed 5
    J, q = w.J[0], w.q[0]
    L = w.L
    with shaken.Shaken(L, 1, w.seed, packed=True, max_records=8) as s:
        s.init(w.init)
        # init stream: sampled rows straight from the oracle's Philox
        sg = s.get_spins(0)[0]
        for r in (0, 1, 12345, L - 1):
            for call in (0, 1, L // 4 - 1):
                n = (r * L) // 4 + call
                want = np.where(so.philox4x32_10((n, 0, 0, 0xFFFFFFFF), (w.seed, 0)) < 2**31, 1, -1)
                assert np.array_equal(sg[r, 4 * call: 4 * call + 4], want)
        s.run(J, q, 2, 1)
        sigma_k = s.get_spins(0)[0].copy()
        t = s.step
        s.run(J, q, 1, 1)
        tau_new = s.get_spins(1)[0]
        sigma_new = s.get_spins(0)[0]
        bands = [(0, 3), (15, 3), (16383, 2), (L - 2, 2), (20000, 1)]   # across task and wrap boundaries
        for r0, n in bands:
            assert np.array_equal(so.half_step_rows(sigma_k, w.seed, 0, J, q, t, 0, r0, n), tau_new[r0:r0 + n]), ("half0", r0)
            assert np.array_equal(so.half_step_rows(tau_new, w.seed, 0, J, q, t, 1, r0, n), sigma_new[r0:r0 + n]), ("half1", r0)
        assert np.array_equal(s.observables()[-1, 0], so.measure(sigma_new, tau_new))


@pytest.mark.parametrize("packed", [False, True])
def test_maximum_lattice_side_65536_sampled_rows(packed):
    """Edge case: the largest L the library accepts (4.3e9 sites per layer; site indices reach 2^32, Philox counter word
    0 reaches 2^30).  One recorded step from an iid start, checked on sampled row bands against the oracle (across strip
    and wrap boundaries) and on the magnetisation sums by brute force."""
    L, seed, J, q = 65536, 9, 0.44, 0.66
    with shaken.Shaken(L, 1, seed, packed=packed, max_records=2) as s:
        s.init(0)
        sigma0 = s.get_spins(0)[0].copy()
        for r in (0, 40000, L - 1):                       # init stream at the far end of the index range
            n = (r * L) // 4 + (L // 4 - 1)
            want = np.where(so.philox4x32_10((n, 0, 0, 0xFFFFFFFF), (seed, 0)) < 2**31, 1, -1)
            assert np.array_equal(sigma0[r, L - 4:], want)
        s.run(J, q, 1, 1)
        tau1 = s.get_spins(1)[0]
        for r0, n in [(0, 2), (L - 2, 2), (33333, 1), (221, 3)]:
            assert np.array_equal(so.half_step_rows(sigma0, seed, 0, J, q, 0, 0, r0, n), tau1[r0:r0 + n]), ("half0", r0)
        del sigma0
        sigma1 = s.get_spins(0)[0]
        for r0, n in [(0, 2), (L - 2, 2), (50001, 1)]:
            assert np.array_equal(so.half_step_rows(tau1, seed, 0, J, q, 0, 1, r0, n), sigma1[r0:r0 + n]), ("half1", r0)
        rec = s.observables()[-1, 0]
        assert rec[0] == int(sigma1.sum(dtype=np.int64)) and rec[1] == int(tau1.sum(dtype=np.int64))
        assert rec[3] == int((sigma1.astype(np.int16) * tau1).sum(dtype=np.int64))          # E_q


def test_cfg2_full_length_10000_steps_against_the_oracle():
    """cfg 2 at full length (SURVEY 8(c) last row: "full-length full-size oracle runs are still the goal for cfg 1-2"):
    10^4 steps of 1024^2 at the honeycomb point, records every 10 steps, in ONE shaken_run call -- one cooperative launch
    of the band kernel with 20 000 stamped hand-overs per band.  The oracle advances half-step by half-step with its row
    function spread over the host cores and takes its six sums every 10 steps; all 1000 records and both final layers
    must agree bit for bit."""
    w = workloads.config(2)
    L, J, q = w.L, w.J[0], w.q[0]
    sigma = np.ones((L, L), dtype=np.int8)
    want = np.zeros((w.n_steps // w.obs_every, 6), dtype=np.int64)
    with ThreadPoolExecutor(rowsplit.n_threads()) as pool:
        for t in range(w.n_steps):
            tau = rowsplit.half_step(sigma, w.seed, 0, J, q, t, 0, pool)
            sigma = rowsplit.half_step(tau, w.seed, 0, J, q, t, 1, pool)
            if (t + 1) % w.obs_every == 0:
                want[(t + 1) // w.obs_every - 1] = so.measure(sigma, tau)
    with shaken.Shaken(L, 1, w.seed, max_records=w.n_steps // w.obs_every) as s:
        s.init(w.init)
        s.run(J, q, w.n_steps, w.obs_every)
        assert s.launch_count == 1                     # the one-launch band path is what ran
        rec = s.observables()
        assert rec.shape == (1000, 1, 6)
        bad = np.nonzero((rec[:, 0] != want).any(axis=1))[0]
        assert bad.size == 0, f"first differing record {bad[:3]}"
        assert np.array_equal(s.get_spins(1)[0], tau) and np.array_equal(s.get_spins(0)[0], sigma)
    # the paper's honeycomb critical point: started from all +1, |m| decays but has not vanished at L = 1024
    assert 0 < abs(int(want[-1, 0])) < L * L


def test_cfg5_packed_32768_whole_lattice_one_step():
    """Every site of one full step at cfg 5's real size (2.1e9 site updates) against the oracle's row function over all
    rows; the record against the oracle's sums of the (already verified) layers."""
    w = workloads.config(5)
    J, q, L = w.J[0], w.q[0], w.L
    with shaken.Shaken(L, 1, w.seed, packed=True, max_records=8) as s:
        s.init(w.init)
        s.run(J, q, 2, 1)
        sigma_k = s.get_spins(0)[0].copy()
        t = s.step
        s.run(J, q, 1, 1)
        tau_new, sigma_new = s.get_spins(1)[0], s.get_spins(0)[0]
        with ThreadPoolExecutor(rowsplit.n_threads()) as pool:
            assert rowsplit.mismatching_rows(sigma_k, tau_new, w.seed, 0, J, q, t, 0, pool) == []
            assert rowsplit.mismatching_rows(tau_new, sigma_new, w.seed, 0, J, q, t, 1, pool) == []
        assert np.array_equal(s.observables()[-1, 0], so.measure(sigma_new, tau_new))


@pytest.mark.skipif(host_memory_gb() < 48, reason="needs about 20 GB of host memory for three 65536^2 int8 layers")
def test_maximum_lattice_side_65536_whole_lattice_one_step_int8():
    """L = 65536 int8 (4.3e9 sites per layer): every row of both half-steps of a recorded step from an iid start."""
    L, seed, J, q = 65536, 9, 0.44, 0.66
    with shaken.Shaken(L, 1, seed, max_records=2) as s:
        s.init(0)
        sigma0 = s.get_spins(0)[0].copy()
        s.run(J, q, 1, 1)
        tau1 = s.get_spins(1)[0]
        with ThreadPoolExecutor(rowsplit.n_threads()) as pool:
            assert rowsplit.mismatching_rows(sigma0, tau1, seed, 0, J, q, 0, 0, pool) == []
            del sigma0
            sigma1 = s.get_spins(0)[0]
            assert rowsplit.mismatching_rows(tau1, sigma1, seed, 0, J, q, 0, 1, pool) == []
        rec = s.observables()[-1, 0]
        assert rec[0] == int(sigma1.sum(dtype=np.int64)) and rec[1] == int(tau1.sum(dtype=np.int64))


@pytest.mark.skipif(host_memory_gb() < 48, reason="needs about 22 GB of host memory")
def test_chain_planes_beyond_4GiB_three_chains_of_49152():
    """Three chains of 49152^2 int8 (2.4 GB per plane): chain 1 straddles the 4 GiB offset, chain 2 starts above it; one
    recorded step with per-chain couplings, sampled row bands of chains 1 and 2 (incl. the row that contains byte offset
    2^32, strip boundaries and the torus wrap) against the oracle, and M_sigma, M_tau of every chain by brute force."""
    L, n, seed = 49152, 3, 13
    J = np.array([0.44, 0.7, 0.3])
    q = np.array([0.66, 0.7, 1.5])
    with shaken.Shaken(L, n, seed, max_records=2) as s:
        s.init(0)
        sigma0 = s.get_spins(0).copy()
        s.run_grid(J, q, 1, 1)
        tau1 = s.get_spins(1)
        row_4g = (2**32 - L * L) // L                 # row of chain 1 that holds byte offset 2^32 of the layer
        for ch in (1, 2):
            for r0, k in [(0, 2), (L - 2, 2), (row_4g - 1, 3), (221, 3), (30011, 1)]:
                assert np.array_equal(so.half_step_rows(sigma0[ch], seed, ch, J[ch], q[ch], 0, 0, r0, k), tau1[ch, r0:r0 + k]), ("half0", ch, r0)
        del sigma0
        sigma1 = s.get_spins(0)
        for ch in (1, 2):
            for r0, k in [(0, 2), (L - 2, 2), (row_4g - 1, 3), (40001, 2)]:
                assert np.array_equal(so.half_step_rows(tau1[ch], seed, ch, J[ch], q[ch], 0, 1, r0, k), sigma1[ch, r0:r0 + k]), ("half1", ch, r0)
        rec = s.observables()[-1]
        for ch in range(n):
            assert rec[ch, 0] == int(sigma1[ch].sum(dtype=np.int64)) and rec[ch, 1] == int(tau1[ch].sum(dtype=np.int64))
