"""Long runs (``-m gpu``): the one-launch kernels (band in both schedules, cluster, alternate band) against the per-half-step strip kernels of
the same library over tens of thousands of steps.  This is NOT an oracle comparison (the oracle is too slow for these
lengths; the strip kernels are compared with it bit for bit elsewhere, and the band kernel over 10^4 steps in
test_gpu_fullsize.py) -- it is a race detector for the hand-over protocols: a stale or torn boundary word anywhere in
10^5 stamped hand-overs per band would change the final configuration."""
import numpy as np
import pytest

from paper_1908_07341_b200 import shaken

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("L,n_chains,steps,alt", [(1024, 1, 40000, False), (512, 1, 40000, False), (768, 1, 20000, False), (512, 3, 30000, False), (2048, 1, 6000, False), (272, 5, 50000, False),
                                                 (64, 1, 100000, False), (128, 2, 50000, False),
                                                 (1024, 1, 30000, True), (272, 3, 50000, True)])
def test_one_launch_kernels_agree_with_the_strip_kernels_over_long_runs(L, n_chains, steps, alt):
    seed = 4000 + L
    J = np.linspace(0.55, 0.7, n_chains)
    q = np.linspace(0.6, 0.7, n_chains)
    obs = max(steps // 50, 1)
    out = []
    for variant in (0, 3):
        with shaken.Shaken(L, n_chains, seed, max_records=64) as s:
            s.set_variant(variant)
            s.init(0)
            l0 = s.launch_count
            for part in (steps // 3, steps - steps // 3):
                if alt:
                    s.run_alternate(J, part, obs)
                else:
                    s.run_grid(J, q, part, obs)
            if variant == 0:
                assert s.launch_count - l0 == 2, "one launch per run call expected on the one-launch paths"
            out.append((s.get_spins(0).copy(), s.get_spins(1).copy() if not alt else None, s.observables().copy()))
    assert np.array_equal(out[0][0], out[1][0]), "sigma differs between the one-launch kernel and the strip kernels"
    if not alt:
        assert np.array_equal(out[0][1], out[1][1]), "tau differs"
    assert np.array_equal(out[0][2], out[1][2]), "records differ"
    assert abs(int(out[0][2][-1, 0, 0])) < L * L     # (not a frozen lattice: the run did something)


@pytest.mark.parametrize("L,steps,obs", [(1024, 4000, 1), (272, 6000, 1), (528, 3000, 2), (144, 5000, 1)])
def test_data_flow_band_kernel_records_on_every_step_over_long_runs(L, steps, obs):
    """kernel_flow.cuh keeps the records in flight in a ring of shared-memory accumulators and lets the last warp that
    delivers its part flush a record: thousands of consecutive recorded steps (groups of warps drifting apart by several
    half-steps) against the strip kernels and the two-phase band kernel."""
    seed = 4100 + L
    out = []
    for variant, two_phase in ((0, 0), (0, 1), (3, 0)):
        with shaken.Shaken(L, 1, seed, max_records=steps // obs + 2) as s:
            s.set_variant(variant)
            s.test_band_hook(2, two_phase)
            s.init(0)
            s.run(0.6585, 0.6585, steps // 2 + 1, obs)
            s.run(0.6585, 0.6585, steps - steps // 2 - 1, obs)
            out.append((s.get_spins(0).copy(), s.get_spins(1).copy(), s.observables().copy()))
    for other in out[1:]:
        for a, b in zip(out[0], other):
            assert np.array_equal(a, b)
    assert len(out[0][2]) == steps // obs
