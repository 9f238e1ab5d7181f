"""Full-size parity (``-m gpu``): BASELINE.json configs 2-5 at their real L and chain count, in the launch
configuration bench.py times.  The oracle is too slow for full-length runs here (SURVEY 8(c) last row), so:

* complete lattices are compared for the first steps, and
* *snapshot induction*: the GPU state after k steps is downloaded, the oracle advances ONE step from it with
  ``step = k`` (legal because the randomness is indexed by the step), and the result must equal the GPU state
  after k+1 steps, spins and records;
* at L = 32768 (cfg 5, 2.1e9 site updates per step) the oracle computes sampled bands of rows of each half-step
  (``oracle.half_step_rows``) from the downloaded source layer, and the six sums by brute force.
"""
import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import shaken, workloads

pytestmark = pytest.mark.gpu


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
