"""Parity (``-m gpu``) of the alternate even/odd heat bath on the square lattice:
libshaken's shaken_run_alternate through the C ABI against the oracle's run_alternate, bit for bit, both layouts."""
import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import sampling, shaken

pytestmark = pytest.mark.gpu


def test_alternate_threshold_tables_are_identical():
    for J in (0.0, 0.1, 0.3, 0.4406867935097715, 0.6, 1.0, 12.0, -0.3):
        assert np.array_equal(shaken.alt_thresholds(J), so.alt_thresholds(J)), J


@pytest.mark.parametrize("L,n_chains,packed,J,init,steps,obs", [
    (16, 1, False, 0.3, 0, 6, 1),          # one vector per row
    (48, 3, False, 0.44, 0, 5, 2),
    (528, 1, False, 0.45, 0, 3, 1),        # 33 vectors per row: ragged last warp trip
    (272, 2, False, 20.0, 0, 4, 1),        # saturated: majority rule + coin flips on ties
    (64, 2, False, 0.0, 1, 3, 1),          # J = 0: coin flips only
    (32, 1, True, 0.3, 0, 6, 1),           # one word per row
    (96, 3, True, 0.44, -1, 5, 2),
    (1056, 1, True, 0.45, 0, 3, 1),        # 33 words per row
    (160, 2, True, -0.3, 0, 4, 1),         # antiferromagnetic sign
])
def test_alternate_runs_match_oracle_bit_for_bit(L, n_chains, packed, J, init, steps, obs):
    seed = 3000 + L
    o = so.Oracle(L, n_chains, seed)
    o.init(init)
    o.run_alternate(J, steps, obs)
    with shaken.Shaken(L, n_chains, seed, packed=packed, max_records=steps) as s:
        s.init(init)
        s.run_alternate(J, steps, obs)
        assert s.step == o.step
        assert np.array_equal(s.get_spins(0), o.get_spins(0)), "sigma differs"
        assert np.array_equal(s.get_spins(1), o.get_spins(1)), "tau must not move"
        assert np.array_equal(s.observables(), o.observables()), "records differ"


@pytest.mark.parametrize("L,n_chains,group", [(16, 3, 1), (32, 6, 2), (64, 2, 1), (128, 3, 3), (48, 8, 4)])
def test_alternate_small_lattice_path_and_per_half_step_kernels_agree_with_oracle(L, n_chains, group):
    """L <= 128 runs in one launch with sigma in shared memory (alt_small_i8); variant 3 forces the per-half-step
    kernels.  Both against the oracle, with per-chain couplings, records every other step and coalescence times."""
    seed, steps = 900 + L, 25
    J = np.repeat(np.linspace(0.15, 0.5, n_chains // group), group)
    o = so.Oracle(L, n_chains, seed)
    o.set_coupling(group)
    o.init(2 if group > 1 else 0)
    o.run_alternate(J, steps, 2)
    for variant in (0, 3):
        with shaken.Shaken(L, n_chains, seed, max_records=steps) as s:
            s.set_variant(variant)
            s.set_coupling(group)
            s.init(shaken.INIT_SANDWICH if group > 1 else 0)
            s.run_alternate(J, 10, 2)
            s.run_alternate(J, steps - 10, 2)
            assert np.array_equal(s.get_spins(0), o.get_spins(0)), variant
            assert np.array_equal(s.observables(), o.observables()), variant
            assert np.array_equal(s.coalescence(), o.coalescence()), variant


def test_alternate_batch_of_mid_size_chains_runs_in_the_one_cta_per_chain_path():
    """80 chains of 208^2 are enough to fill the machine, so the run takes the shared-memory path (one launch) although
    L > 128; variant 3 takes the per-half-step kernels (13 vectors per row: the generic form).  Both against the oracle."""
    L, n_chains, seed, steps = 208, 80, 77, 4
    J = np.linspace(0.2, 0.6, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_alternate(J, steps, 2)
    for variant, launches in ((0, 1), (3, 2 * steps)):
        with shaken.Shaken(L, n_chains, seed, max_records=steps) as s:
            s.set_variant(variant)
            s.init(0)
            l0 = s.launch_count
            s.run_alternate(J, steps, 2)
            assert s.launch_count - l0 == launches
            assert np.array_equal(s.get_spins(0), o.get_spins(0)), variant
            assert np.array_equal(s.observables(), o.observables()), variant


@pytest.mark.parametrize("L,n_chains", [(144, 1), (160, 74), (272, 3), (304, 37), (528, 1), (784, 2), (1024, 1), (2048, 1), (1024, 4)])
def test_alternate_band_path_one_launch_per_run_matches_oracle(L, n_chains):
    """128 < L <= 2048 with few chains: the whole shaken_run_alternate call is ONE cooperative launch (alt_band_i8: row
    bands in shared memory, two halo rows per side, one hand-over per full step).  Per-chain couplings, records on some
    steps only, the run split in the middle of a recording interval; the same run through the per-half-step kernels
    (variant 3) must give the same bits."""
    seed, steps = 500 + L, 9
    J = np.linspace(0.25, 0.6, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_alternate(J, steps, 2)
    for variant in (0, 3):
        with shaken.Shaken(L, n_chains, seed, max_records=steps) as s:
            s.set_variant(variant)
            s.init(0)
            l0 = s.launch_count
            s.run_alternate(J, 5, 2)
            s.run_alternate(J, steps - 5, 2)
            if variant == 0:
                assert s.launch_count - l0 == 2, "one cooperative launch per run call expected"
            assert s.step == o.step
            assert np.array_equal(s.get_spins(0), o.get_spins(0)), f"sigma differs, variant {variant}"
            assert np.array_equal(s.observables(), o.observables()), f"records differ, variant {variant}"


@pytest.mark.parametrize("alternate", [False, True])
def test_band_path_stamp_wrap_and_refused_cooperative_launch(alternate):
    """Two corners of the one-launch band path, through the test hook: (i) the 32-bit stamp counter of the hand-over
    buffer about to wrap -- the buffer is cleared and the stamps restart; (ii) a refused cooperative launch -- the same
    call falls back to the per-half-step kernels.  Both in the middle of a run, results unchanged."""
    L, seed = 528, 61
    o = so.Oracle(L, 1, seed)
    o.init(0)
    if alternate:
        o.run_alternate(0.44, 12, 3)
    else:
        o.run(0.5, 0.7, 12, 3)
    with shaken.Shaken(L, 1, seed, max_records=8) as s:
        run = (lambda n: s.run_alternate(0.44, n, 3)) if alternate else (lambda n: s.run(0.5, 0.7, n, 3))
        s.init(0)
        l0 = s.launch_count
        run(4)                                          # band kernel, stamps 1 .. 4
        assert s.launch_count - l0 == 1
        s.test_band_hook(0, 2**32 - 4)                  # the next launch would need stamps beyond 2^32 - 1
        run(3)
        assert s.launch_count - l0 == 2
        s.test_band_hook(1, 1)                          # refuse the next cooperative launch
        l1 = s.launch_count
        run(2)
        assert s.launch_count - l1 >= 4, "per-half-step kernels expected after the refusal"
        run(3)                                          # band kernel again
        assert s.step == o.step
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.get_spins(1), o.get_spins(1))
        assert np.array_equal(s.observables(), o.observables())


def test_alternate_grid_of_couplings_resume_and_chain_offset():
    L, n_chains, seed = 80, 5, 41
    J = np.array([0.1, 0.3, 0.44, 0.6, 0.9])
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_alternate(J, 7, 1)
    for packed in (False,):
        with shaken.Shaken(L, n_chains, seed, packed=packed, max_records=16) as s:
            s.init(0)
            s.run_alternate(J, 3, 1)                               # split runs: the step counter drives the randomness
            s.run_alternate(J, 4, 1)
            assert np.array_equal(s.get_spins(0), o.get_spins(0))
            assert np.array_equal(s.observables(), o.observables())
        with shaken.Shaken(L, 2, seed, packed=packed) as part:     # chains 3, 4 of the batch alone
            part.set_chain_offset(3)
            part.init(0)
            part.run_alternate(J[3:], 7, 0)
            assert np.array_equal(part.get_spins(0), o.get_spins(0)[3:])
    # the shaken dynamics and the alternate one can be mixed on one context: both only advance the step counter
    o.run(0.3, 0.5, 2, 1)
    o.run_alternate(0.35, 2, 1)
    with shaken.Shaken(L, n_chains, seed, max_records=16) as s:
        s.init(0)
        s.run_alternate(J, 7, 1)
        s.run(0.3, 0.5, 2, 1)
        s.run_alternate(0.35, 2, 1)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.get_spins(1), o.get_spins(1))
        assert np.array_equal(s.observables(), o.observables())


@pytest.mark.parametrize("packed", [False, True])
def test_alternate_coupled_pairs_coalescence_and_exact_sampling(packed):
    L, n_pairs, seed = 32, 8, 19
    J = np.repeat(np.linspace(0.1, 0.38, n_pairs), 2)
    o = so.Oracle(L, 2 * n_pairs, seed)
    o.set_coupling(2)
    o.init(2)
    with shaken.Shaken(L, 2 * n_pairs, seed, packed=packed) as s:
        s.set_coupling(2)
        s.init(shaken.INIT_SANDWICH)
        for chunk in (1, 30, 60):
            o.run_alternate(J, chunk, 0)
            s.run_alternate(J, chunk, 0)
            assert np.array_equal(s.coalescence(), o.coalescence()), chunk
        sig = s.get_spins(0)
        assert np.array_equal(sig, o.get_spins(0))
        assert np.all(sig[0::2] >= sig[1::2])                      # attractive: the order is preserved
        assert np.any(s.coalescence() > 0)
        # Propp-Wilson draws from the square-lattice Gibbs measure, driver against driver
        Jl = np.repeat(np.linspace(0.1, 0.3, n_pairs), 2)
        want, T_want = so.propp_wilson(o, Jl, None, base=1 << 34)
        got, T = sampling.propp_wilson(s, Jl, None, base=1 << 34)
        assert T == T_want and np.array_equal(got, want)


def test_alternate_full_size_rows_against_the_oracle():
    """cfg 4 size (L = 16384, int8) and cfg 5 size (L = 8192 x 4 chains, packed): one half-step each way on random
    spins, sampled row windows (first, last, across the middle) recomputed by the oracle's context-free row function,
    and the record of the step against sums taken with numpy from the downloaded spins."""
    for L, n_chains, packed in ((16384, 1, False), (8192, 4, True)):
        seed, J, t0 = 7, 0.44, 5
        with shaken.Shaken(L, n_chains, seed, packed=packed, max_records=4) as s:
            s.init(0)
            s.step = t0
            before = s.get_spins(0)
            s.run_alternate(J, 1, 1)
            after = s.get_spins(0)
            rec = s.observables()
            ch = n_chains - 1
            # the oracle needs the state between the half-steps: rows of half 1 depend on rows r-1 .. r+1 after half 0
            for r0, n in ((0, 3), (L - 3, 3), (L // 2 - 1, 4), (4097, 2)):
                lo, hi = r0 - 1, r0 + n + 1                        # window of half-0 rows needed (may wrap)
                rows = [(r % L) for r in range(lo, hi)]
                mid = np.array(before[ch])                         # only the window rows are brought to half-0 state
                for r in rows:
                    mid[r] = so.alt_half_step_rows(before[ch], seed, ch, J, t0, 0, r, 1)[0]
                want = so.alt_half_step_rows(mid, seed, ch, J, t0, 1, r0, n)
                assert np.array_equal(after[ch, r0:r0 + n], want), (L, r0)
            x = after[ch].astype(np.int32)
            assert rec[0, ch, 0] == int(x.sum(dtype=np.int64))
            assert rec[0, ch, 4] == int((x * np.roll(x, -1, 1)).sum(dtype=np.int64))
            assert rec[0, ch, 5] == int((x * np.roll(x, -1, 0)).sum(dtype=np.int64))
            assert np.all(rec[0, :, 1:4] == 0)


def test_alternate_error_paths_and_bookkeeping():
    with shaken.Shaken(32, 2, 1, max_records=3) as s:
        s.init(1)
        for bad in (float("nan"), float("inf")):
            with pytest.raises(shaken.ShakenError) as ei:
                s.run_alternate(bad, 1, 0)
            assert ei.value.code == shaken.EINVAL
        with pytest.raises(shaken.ShakenError):
            s.run_alternate(0.3, -1, 0)
        with pytest.raises(ValueError):
            s.run_alternate([0.3, 0.3, 0.3], 1, 0)                  # one J per chain
        assert s.step == 0 and s.observables().shape[0] == 0        # nothing ran
        s.run_alternate(0.3, 0, 1)
        assert s.step == 0
        l0 = s.launch_count
        s.run_alternate(0.3, 7, 3)                                  # records after global steps 3 and 6
        assert s.step == 7 and s.observables().shape[0] == 2 and s.launch_count == l0 + 1
        rec = s.observables()
        assert np.all(np.abs(rec[:, :, 0]) <= 32 * 32) and np.all(rec[:, :, 0] % 2 == 0)
        s.run_alternate(20.0, 2, 2)                                 # step 8 is recorded
        assert s.observables().shape[0] == 3
        before = s.get_spins(0).copy()
        with pytest.raises(shaken.ShakenError) as ei:
            s.run_alternate(0.3, 1, 1)                              # bound record buffer (3 records) is full
        assert ei.value.code == shaken.ENOSPC
        assert s.step == 9 and np.array_equal(s.get_spins(0), before)
    with shaken.Shaken(32, 1, 1, max_records=3) as s:               # all +1 at J = 20 stays all +1: M = L^2, C_x = C_y = L^2
        s.init(1)
        s.run_alternate(20.0, 3, 1)
        assert np.array_equal(s.observables()[:, 0], np.tile([1024, 0, 0, 0, 1024, 1024], (3, 1)))
