"""Parity tests proper (``-m gpu``): the CUDA path, called through the C ABI, against the CPU oracle on the same
seeded inputs -- bit-exact spins and int64 records, derived doubles within 1e-12 relative (BASELINE.json).

Sizes are chosen so the oracle finishes in seconds while the lattice still spans several warp strips, several
row blocks and a ragged tail (L/16 not a multiple of 32).  Full-size checks are in test_gpu_fullsize.py."""
import ctypes as C
import math
import os

import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import shaken, workloads
from tests import conftest

pytestmark = pytest.mark.gpu

REL = 1e-12   # BASELINE.json north_star: derived double-precision quantities agree within 1e-12 relative


def assert_same_state(s: shaken.Shaken, o: so.Oracle, what=""):
    assert s.step == o.step, what
    assert np.array_equal(s.get_spins(0), o.get_spins(0)), f"sigma differs {what}"
    assert np.array_equal(s.get_spins(1), o.get_spins(1)), f"tau differs {what}"
    assert np.array_equal(s.observables(), o.observables()), f"records differ {what}"


# ----------------------------------------------------------------------------- RNG
def test_device_philox_matches_curand_device_function_and_oracle():
    """Third-party pin on the GPU box: cuRAND's device function curand_Philox4x32_10 (all four counter words and
    both key words free) against the library's Philox AND the oracle's, 2^20 random (counter, key) pairs plus
    edge patterns.  This is the pin for counter word 3, which cuRAND's host generator cannot reach."""
    path = conftest.build_curand_ref()
    assert path and os.path.exists(path), "tests/libcurandref.so missing (nvcc needed)"
    ref = C.CDLL(path)
    ref.curand_ref_philox.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_longlong]
    ref.curand_ref_philox.restype = C.c_int
    rng = np.random.default_rng(2024)
    n = 1 << 20
    ctr = rng.integers(0, 2**32, size=(n, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2**32, size=(n, 2), dtype=np.uint64).astype(np.uint32)
    edge = np.array([[0, 0, 0, 0], [0xFFFFFFFF] * 4, [1, 0, 0, 0], [0, 0, 0, 1], [0, 0, 5, 0xFFFFFFFF], [7, 2, 0, 0xFFFFFFFF]],
                    dtype=np.uint32)
    ctr[: len(edge)] = edge
    key[:3] = [[0, 0], [0xFFFFFFFF, 0xFFFFFFFF], [1, 0]]
    want = np.empty_like(ctr)
    assert ref.curand_ref_philox(ctr.ctypes.data, key.ctypes.data, want.ctypes.data, n) == 0
    got = shaken.philox_words(ctr, key)
    assert np.array_equal(got, want)
    for i in list(range(64)) + list(rng.integers(0, n, size=2000)):
        assert np.array_equal(so.philox4x32_10(ctr[i], key[i]), want[i]), i


def test_threshold_tables_of_library_and_oracle_are_identical():
    """SURVEY 8(c) point 7: the two sides evaluate exp() with the same libm here, but diff the tables anyway."""
    J, q = workloads.grid_couplings()
    for a, b in list(zip(J, q)) + [(0.5, 0.5), (0.6585, 0.6585), (0.7, 0.7), (0.45, 10.0), (0.44, 0.66), (-0.2, 0.3)]:
        assert np.array_equal(shaken.thresholds(a, b), so.thresholds(a, b)), (a, b)


# ----------------------------------------------------------------------------- int8 layout
@pytest.mark.parametrize("L,n_chains,J,q,init,steps,obs", [
    (16, 1, 0.5, 0.5, 0, 5, 1),          # smallest lattice: one 16-byte vector per row
    (48, 2, 0.3, 1.1, 0, 6, 2),          # 3 lanes of a warp active
    (64, 1, 0.5, 0.5, 0, 50, 1),         # cfg 1 shape
    (528, 1, 0.6585, 0.6585, 1, 4, 1),   # 33 vectors per row: two strips, ragged tail; all +1 start
    (1024, 1, 0.44, 0.66, -1, 3, 3),     # the paper's benchmark couplings, all -1 start (:200)
    (272, 3, 0.45, 10.0, 0, 5, 1),       # saturated thresholds (cfg 5 couplings)
    (64, 2, 0.0, 0.0, 1, 3, 1),          # J = q = 0: pure coin flips
    (64, 1, -0.4, 0.7, 0, 4, 1),         # antiferromagnetic J (threshold order reversed)
])
def test_int8_runs_match_oracle_bit_for_bit(L, n_chains, J, q, init, steps, obs):
    seed = 1000 + L
    o = so.Oracle(L, n_chains, seed)
    o.init(init)
    o.run(J, q, steps, obs)
    with shaken.Shaken(L, n_chains, seed, packed=False, max_records=steps) as s:
        s.init(init)
        s.run(J, q, steps, obs)
        assert_same_state(s, o, f"L={L}")


@pytest.mark.parametrize("L,n_chains,J,q,init,steps,obs", [
    (32, 1, 0.5, 0.5, 0, 5, 1),          # one word per row
    (96, 2, 0.3, 1.1, 0, 6, 2),          # 3 words per row
    (1056, 1, 0.45, 10.0, 0, 3, 1),      # 33 words per row: two strips, ragged tail; cfg 5 couplings
    (256, 3, 0.6585, 0.6585, -1, 5, 1),
    (64, 1, -0.4, 0.7, 0, 4, 1),
])
def test_packed_runs_match_oracle_bit_for_bit(L, n_chains, J, q, init, steps, obs):
    seed = 2000 + L
    o = so.Oracle(L, n_chains, seed)
    o.init(init)
    o.run(J, q, steps, obs)
    with shaken.Shaken(L, n_chains, seed, packed=True, max_records=steps) as s:
        s.init(init)
        s.run(J, q, steps, obs)
        assert_same_state(s, o, f"packed L={L}")


def test_int8_and_packed_layouts_give_identical_spins_and_records():
    L, n_chains, seed = 160, 2, 9
    outs = []
    for packed in (False, True):
        with shaken.Shaken(L, n_chains, seed, packed=packed, max_records=8) as s:
            s.init(0)
            s.run(0.4, 0.8, 7, 1)
            outs.append((s.get_spins(0), s.get_spins(1), s.observables()))
    for a, b in zip(*outs):
        assert np.array_equal(a, b)


# ----------------------------------------------------------------------------- batched chains, grids
def test_grid_of_couplings_matches_oracle_and_chains_are_independent():
    """cfg 3 shape at reduced size: per-chain (J, q) tables, 4 replicas per point share couplings but not
    randomness; chain c of a batch equals the same chain index run alone (counter word 1 = chain)."""
    L, seed = 64, 11
    J, q = workloads.grid_couplings()
    J, q = np.array(J[::16]), np.array(q[::16])          # 32 chains across the whole grid incl. q = 10, 20
    n = len(J)
    o = so.Oracle(L, n, seed)
    o.init(0)
    o.run_grid(J, q, 12, 1)
    with shaken.Shaken(L, n, seed, max_records=12) as s:
        s.init(0)
        s.run_grid(J, q, 12, 1)
        assert_same_state(s, o, "grid")
        rec = s.observables()
    with shaken.Shaken(L, n, seed, packed=True, max_records=12) as s:
        s.init(0)
        s.run_grid(J, q, 12, 1)
        assert_same_state(s, o, "grid packed")
    # derived statistics (a9) within 1e-12 relative of the oracle's
    for ch in (0, 7, 31):
        a = shaken.derived_stats(rec[2:, ch, 0], L * L)
        b = so.derived_stats(o.observables()[2:, ch, 0], L * L)
        for k in ("m", "abs_m", "m2", "m4", "var_m", "binder"):
            assert a[k] == b[k] or abs(a[k] - b[k]) <= REL * abs(b[k]), (ch, k, a[k], b[k])
        e1 = shaken.energy(J[ch], q[ch], rec[-1, ch, 2], rec[-1, ch, 3])
        e2 = so.energy(J[ch], q[ch], o.observables()[-1, ch, 2], o.observables()[-1, ch, 3])
        assert abs(e1 - e2) <= REL * abs(e2)


def test_batch_sharded_over_two_contexts_equals_the_single_batch():
    """a batch split into per-rank contexts with shaken_set_chain_offset is bit-identical to
    the single batch (here both 'ranks' run one after the other on the one GPU; no kernel waits on another)."""
    from paper_1908_07341_b200 import parallel

    L, n, seed, steps = 128 + 16, 5, 29, 7                # above the small-lattice path, ragged strip
    J = np.array([0.2, 0.45, 0.7, 0.05, 1.1])
    q = np.array([0.3, 10.0, 0.7, 2.0, 0.1])
    o = so.Oracle(L, n, seed)
    o.init(0)
    o.run_grid(J, q, steps, 1)
    want_rec, want_sigma = o.observables(), o.get_spins(0)
    for packed in (False,) if L % 32 else (False, True):
        for world in (2, 3):
            for rank in range(world):
                first, count = parallel.chain_shard(n, world, rank)
                Jl, ql = parallel.shard_couplings(J, q, world, rank)
                with parallel.open_shard(L, n, seed, world, rank, packed=packed, max_records=steps) as s:
                    s.init(0)
                    s.run_grid(Jl, ql, steps, 1)
                    assert np.array_equal(s.observables(), want_rec[:, first:first + count]), (world, rank)
                    assert np.array_equal(s.get_spins(0), want_sigma[first:first + count]), (world, rank)


def test_run_is_resumable_and_step_counter_drives_the_randomness():
    """run(a); run(b) == run(a+b) bit for bit; set_step + set_spins restores a checkpoint."""
    L, seed, J, q = 96, 5, 0.5, 0.4
    with shaken.Shaken(L, 2, seed, max_records=16) as a, shaken.Shaken(L, 2, seed, max_records=16) as b:
        a.init(0)
        b.init(0)
        a.run(J, q, 9, 3)
        b.run(J, q, 4, 3)
        b.run(J, q, 5, 3)
        assert np.array_equal(a.get_spins(0), b.get_spins(0)) and np.array_equal(a.get_spins(1), b.get_spins(1))
        assert np.array_equal(a.observables(), b.observables()) and a.num_records == 3 and a.step == 9
        # checkpoint: copy state of a into a fresh context, continue both
        with shaken.Shaken(L, 2, seed, use_torch=False) as c:
            c.set_spins(0, a.get_spins(0))
            c.set_spins(1, a.get_spins(1))
            c.step = a.step
            a.run(J, q, 3, 0)
            c.run(J, q, 3, 0)
            assert np.array_equal(a.get_spins(0), c.get_spins(0)) and np.array_equal(a.get_spins(1), c.get_spins(1))
        # a different seed (either key word) changes the trajectory
        for other in (seed + 1, seed + (1 << 32)):
            with shaken.Shaken(L, 2, other) as d:
                d.init(1)
                d.run(J, q, 1, 0)
                with shaken.Shaken(L, 2, seed) as e:
                    e.init(1)
                    e.run(J, q, 1, 0)
                    assert not np.array_equal(d.get_spins(0), e.get_spins(0))


def test_large_step_index_uses_both_counter_words():
    """g = 2t + half spills into counter word 3 when t >= 2^31."""
    L, seed = 32, 3
    t0 = (1 << 31) - 2
    o = so.Oracle(L, 1, seed)
    o.init(0)
    o.step = t0
    o.run(0.5, 0.5, 4, 1)
    for packed in (False, True):
        with shaken.Shaken(L, 1, seed, packed=packed, max_records=4) as s:
            s.init(0)
            s.step = t0
            s.run(0.5, 0.5, 4, 1)
            assert_same_state(s, o, "large t")


def test_state_io_roundtrip_and_validation():
    rng = np.random.default_rng(0)
    for packed, L in ((False, 48), (True, 96)):
        with shaken.Shaken(L, 2, 1, packed=packed) as s:
            x = rng.choice(np.array([-1, 1], dtype=np.int8), size=(2, L, L))
            y = rng.choice(np.array([-1, 1], dtype=np.int8), size=(2, L, L))
            s.set_spins(0, x)
            s.set_spins(1, y)
            assert np.array_equal(s.get_spins(0), x) and np.array_equal(s.get_spins(1), y)
            bad = x.copy()
            bad[1, 3, 5] = 0
            with pytest.raises(shaken.ShakenError) as ei:
                s.set_spins(0, bad)
            assert ei.value.code == shaken.EINVAL
            bad[1, 3, 5] = 3
            with pytest.raises(shaken.ShakenError):
                s.set_spins(1, bad)


def test_observables_on_known_configurations_and_record_bookkeeping():
    """All +1 start, frozen couplings: M = L^2, E_q = L^2, E_J = C_x + C_y = 2 L^2 on every record."""
    L = 64
    for packed in (False, True):
        with shaken.Shaken(L, 1, 4, packed=packed, use_torch=False) as s:
            s.init(1)
            s.run(0.0, 30.0, 3, 1)          # q = 30: T saturated, each half-step copies the other layer
            rec = s.observables()
            assert rec.shape == (3, 1, 6)
            N = L * L
            # flip probability 2^-32 per site per half-step: the all +1 state survives 3 steps
            assert np.array_equal(rec[:, 0], np.array([[N, N, 2 * N, N, N, N]] * 3))
            s.clear_records()
            assert s.num_records == 0
            s.run(0.0, 30.0, 2, 2)
            assert s.num_records == 1 and s.step == 5
            s.init(-1)
            assert s.step == 0 and s.num_records == 0
            s.run(0.0, 30.0, 1, 1)
            assert np.array_equal(s.observables()[0, 0], np.array([-N, -N, 2 * N, N, N, N]))


def test_bound_record_buffer_reports_enospc_before_doing_any_work():
    with shaken.Shaken(32, 1, 1, max_records=2) as s:
        s.init(0)
        s.run(0.5, 0.5, 2, 1)
        before = s.get_spins(0).copy()
        with pytest.raises(shaken.ShakenError) as ei:
            s.run(0.5, 0.5, 1, 1)
        assert ei.value.code == shaken.ENOSPC
        assert s.step == 2 and np.array_equal(s.get_spins(0), before)
        s.run(0.5, 0.5, 3, 0)                 # no records wanted: fine
        assert s.step == 5


def test_records_against_brute_force_from_downloaded_spins():
    """Third implementation of the six sums (numpy roll) on the GPU's own final state."""
    from tests import pins

    L = 112
    with shaken.Shaken(L, 2, 8, max_records=4) as s:
        s.init(0)
        s.run(0.6, 0.3, 4, 4)
        rec = s.observables()
        sg, ta = s.get_spins(0), s.get_spins(1)
        for ch in range(2):
            assert np.array_equal(rec[0, ch], pins.brute_observables(sg[ch], ta[ch]))


def test_cfg1_full_length():
    """BASELINE.json configs[0], complete: L=64, J=q=0.5, iid start, seed 1, 1000 steps, records every step."""
    w = workloads.config(1)
    o = so.Oracle(w.L, 1, w.seed)
    o.init(w.init)
    o.run(w.J[0], w.q[0], w.n_steps, w.obs_every)
    with shaken.Shaken(w.L, 1, w.seed, max_records=w.n_steps) as s:
        s.init(w.init)
        s.run(w.J[0], w.q[0], w.n_steps, w.obs_every)
        assert_same_state(s, o, "cfg1")
        a = shaken.derived_stats(s.observables()[:, 0, 0], w.n_sites)
        b = so.derived_stats(o.observables()[:, 0, 0], w.n_sites)
        for k in a:
            assert a[k] == b[k] or abs(a[k] - b[k]) <= REL * abs(b[k])


@pytest.mark.parametrize("L,n_chains", [(16, 1), (48, 3), (64, 2), (128, 2)])
def test_small_lattice_path_and_generic_kernels_both_match_oracle(L, n_chains):
    """L <= 128 runs in the one-CTA-per-chain persistent kernel (kernel_small.cuh) under variant 0; variants 3 and 8
    force the strip kernels (block tasks / per-warp task lists, include/shaken.h).  All must equal the oracle, records
    included, also when a run is split and obs_every does not divide the split."""
    seed = 77 + L
    J = np.linspace(0.2, 0.9, n_chains)
    q = np.linspace(1.5, 0.1, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_grid(J, q, 11, 3)
    for variant in (0, 3, 8):
        with shaken.Shaken(L, n_chains, seed, max_records=8) as s:
            s.set_variant(variant)
            s.init(0)
            s.run_grid(J, q, 4, 3)
            s.run_grid(J, q, 7, 3)
            assert_same_state(s, o, f"L={L} variant={variant}")


@pytest.mark.parametrize("L,n_chains", [(32, 1), (64, 1), (80, 3), (128, 1), (128, 18), (64, 19), (32, 82), (32, 83), (64, 64), (64, 65),
                                        (128, 28), (128, 29), (128, 56), (128, 57), (64, 92), (64, 93), (112, 40), (48, 150)])
def test_cluster_path_for_few_small_chains_and_one_sm_path_for_many(L, n_chains):
    """Small chains (32 <= L <= 128) run one chain per CLUSTER of 8 SMs while the machine is not full (kernel_cluster.cuh: rows in
    the shared memory of 8 CTAs, neighbour rows through distributed shared memory, fused sums; up to max(18, 100 - 9 L / 16)
    chains, 28 more when records are taken on every or every other step: 82 / 110 at L = 32, 64 / 92 at 64, 28 / 56 at 128), larger batches one chain per SM (kernel_small.cuh): both sides of the
    switch.  Per-chain couplings, records on some steps only and on every step, split runs, a record on the very
    last step of a call (its C_x, C_y are closed from the final sigma)."""
    seed = 300 + L + n_chains
    J = np.linspace(0.3, 0.8, n_chains)
    q = np.linspace(1.1, 0.2, n_chains)
    for obs in (1, 3):
        o = so.Oracle(L, n_chains, seed)
        o.init(0)
        o.run_grid(J, q, 12, obs)
        with shaken.Shaken(L, n_chains, seed, max_records=16) as s:
            s.init(0)
            l0 = s.launch_count
            s.run_grid(J, q, 5, obs)
            s.run_grid(J, q, 4, obs)
            s.run_grid(J, q, 3, obs)
            assert s.launch_count - l0 == 3
            assert_same_state(s, o, f"L={L} chains={n_chains} obs={obs}")


@pytest.mark.parametrize("L,n_chains", [(80, 160), (96, 150), (112, 150), (128, 149), (160, 150), (208, 150), (224, 150)])
def test_one_sm_kernel_block_sizes_for_batches_larger_than_the_machine(L, n_chains):
    """kernel_small.cuh with more chains than SMs: the host picks blocks of 192, 224 or 256 threads (two or three resident CTAs
    per SM, last trip well filled) where two CTAs fit an SM, 512 otherwise; several trips per thread, ragged last trips."""
    J = np.linspace(0.3, 0.8, n_chains)
    q = np.linspace(1.0, 0.2, n_chains)
    o = so.Oracle(L, n_chains, 5)
    o.init(0)
    o.run_grid(J, q, 3, 1)
    with shaken.Shaken(L, n_chains, 5, max_records=4) as s:
        s.init(0)
        s.run_grid(J, q, 2, 1)
        s.run_grid(J, q, 1, 1)
        assert s.launch_count == 3, "init + one launch per run call expected"
        assert_same_state(s, o, f"L={L} chains={n_chains}")


@pytest.mark.parametrize("calls,obs", [((64,), 1), ((65,), 1), ((63, 1, 1), 1), ((128, 1), 1), ((129,), 1), ((130, 61), 3), ((127, 2, 70), 2),
                                       ((200,), 1)])
def test_cluster_kernel_record_ring_boundaries(calls, obs):
    """The cluster kernel collects a CTA's partial sums in a shared-memory ring of 64 records and adds it to the records in
    global memory when it is full and at the end of a launch: runs whose record counts end just before, on and just after a
    multiple of 64, with and without a record on the very last step of a call, against the oracle."""
    L, n_chains, seed, J, q = 64, 2, 77, 0.5, 0.6
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    with shaken.Shaken(L, n_chains, seed, max_records=sum(calls) // obs + 2) as s:
        s.init(0)
        for n in calls:
            o.run(J, q, n, obs)
            s.run(J, q, n, obs)
            assert_same_state(s, o, f"calls={calls} obs={obs} after {n}")


@pytest.mark.parametrize("variant", [0, 3, 8])
def test_every_int8_code_path_matches_oracle_on_a_ragged_lattice(variant):
    """L = 272: 17 vectors per row (ragged warp strip), several row blocks per chain, three chains with different
    couplings incl. a saturated table; records on some steps only, so launches with and without fused sums, the
    deferred bond sums and the closing read-only pass all occur."""
    L, n, seed = 272, 3, 41
    J = np.array([0.44, 0.7, 0.05])
    q = np.array([0.66, 0.7, 20.0])
    o = so.Oracle(L, n, seed)
    o.init(0)
    o.run_grid(J, q, 9, 2)
    with shaken.Shaken(L, n, seed, max_records=8) as s:
        s.set_variant(variant)
        s.init(0)
        s.run_grid(J, q, 5, 2)
        s.run_grid(J, q, 4, 2)
        assert_same_state(s, o, f"variant={variant}")


@pytest.mark.parametrize("L,packed,variant", [(272, False, 0), (528, False, 3), (1056, True, 0), (64, False, 0)])
def test_step_index_crossing_2_to_31_in_every_kernel_family(L, packed, variant):
    """Global step index t0 = 2^31 - 2: g = 2t + half crosses 2^32 inside the run, so counter word 3 (g hi) changes
    between two steps.  L = 272 takes the band kernel (device_half_step_keys), 528 with the strip switch the strip
    kernels (make_step_keys on the host), 1056 the packed kernel, 64 the small-lattice kernel.  Oracle: same t0."""
    seed, t0 = 19, 2**31 - 2
    o = so.Oracle(L, 1, seed)
    o.init(0)
    o.step = t0
    o.run(0.5, 0.8, 4, 1)
    with shaken.Shaken(L, 1, seed, packed=packed, max_records=8) as s:
        s.set_variant(variant)
        s.init(0)
        s.step = t0
        s.run(0.5, 0.8, 3, 1)
        s.run(0.5, 0.8, 1, 1)
        assert s.step == t0 + 4
        assert_same_state(s, o, f"L={L} packed={packed}")


@pytest.mark.parametrize("L,n_chains", [(2048, 1), (1024, 4), (1488, 2)])
def test_band_kernel_tall_bands_per_chain_tables_and_split_runs(L, n_chains):
    """The band kernel's tall-band branch (more than three trips of vectors per band: one chain at L >= ~1792, or four
    chains of 1024^2), with per-chain (J, q) tables, records on some steps only, and the run split over two shaken_run
    calls in the middle of a recording interval (stamp continuity, the pending C_x, C_y of the last record)."""
    seed = 3 + L
    J = np.linspace(0.3, 0.9, n_chains)
    q = np.linspace(1.2, 0.2, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_grid(J, q, 7, 3)
    with shaken.Shaken(L, n_chains, seed, max_records=4) as s:
        s.init(0)
        s.run_grid(J, q, 4, 3)
        s.run_grid(J, q, 3, 3)
        assert s.launch_count == 3, "init + one cooperative launch per run call expected"
        assert_same_state(s, o, f"L={L} chains={n_chains}")


@pytest.mark.parametrize("L,n_chains,steps,obs", [(144, 1, 9, 1), (144, 5, 6, 2), (160, 148, 3, 1), (272, 2, 11, 3), (400, 3, 7, 0),
                                                 (528, 1, 9, 1), (784, 1, 8, 1), (1024, 1, 12, 1), (1040, 2, 5, 2), (1536, 1, 4, 1),
                                                 (1552, 1, 3, 1), (2048, 1, 3, 1), (304, 37, 4, 1)])
@pytest.mark.parametrize("two_phase", [0, 1])
def test_band_kernel_sweep_of_shapes_matches_oracle(L, n_chains, steps, obs, two_phase):
    """The one-launch band path over the shapes it serves: 9 to 128 vectors per row, one-row bands (148 chains), bands of
    28 rows, a ragged last band, several chains with their own couplings, every record cadence; each run split in two.
    Bands of at most seven rows run the data-flow schedule (kernel_flow.cuh: one, two or three warps per row, a second
    warp with a single active lane at L = 528 ...); two_phase = 1 forces the two-phase kernel for them as well."""
    if n_chains * L * L > 4.5e6:
        pytest.skip("beyond the band path")
    seed = 1000 + L + n_chains
    J = np.linspace(0.35, 0.75, n_chains)
    q = np.linspace(0.9, 0.3, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_grid(J, q, steps, obs)
    with shaken.Shaken(L, n_chains, seed, max_records=steps) as s:
        s.test_band_hook(2, two_phase)
        s.init(0)
        l0 = s.launch_count
        s.run_grid(J, q, steps // 2, obs)
        s.run_grid(J, q, steps - steps // 2, obs)
        assert s.launch_count - l0 == 2, "one cooperative launch per run call expected"
        assert_same_state(s, o, f"L={L} chains={n_chains}")


@pytest.mark.parametrize("L,n_chains,packed,variant,steps,obs", [
    (16, 7, False, 8, 6, 1), (48, 5, False, 8, 5, 2), (144, 4, False, 8, 5, 1), (528, 3, False, 8, 4, 1), (1040, 2, False, 8, 3, 0),
    (272, 6, False, 3, 5, 3), (1040, 1, False, 3, 4, 1), (96, 9, False, 3, 4, 1),
    (64, 5, True, 0, 6, 1), (544, 2, True, 0, 4, 2), (1056, 3, True, 0, 3, 1)])
def test_strip_kernels_sweep_of_shapes_matches_oracle(L, n_chains, packed, variant, steps, obs):
    """The per-half-step strip kernels over a sweep of shapes: per-warp ranges that cross chain boundaries (rows narrower and
    wider than a warp strip, ragged last ranges), block tasks, the packed layout; per-chain couplings, every record cadence,
    each run split in two."""
    seed = 2000 + L + 7 * n_chains
    J = np.linspace(0.25, 0.85, n_chains)
    q = np.linspace(1.0, 0.15, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    o.run_grid(J, q, steps, obs)
    with shaken.Shaken(L, n_chains, seed, packed=packed, max_records=steps) as s:
        s.set_variant(variant)
        s.init(0)
        s.run_grid(J, q, steps - steps // 2, obs)
        s.run_grid(J, q, steps // 2, obs)
        assert_same_state(s, o, f"L={L} chains={n_chains} packed={packed} variant={variant}")


@pytest.mark.parametrize("L,n_chains", [(64, 1), (128, 3), (272, 2), (1024, 1), (48, 30)])
def test_single_step_calls_with_a_record_on_every_step(L, n_chains):
    """shaken_run(1) over and over with a record each time: every call is one launch of a one-launch kernel (cluster, band
    or one-SM) whose only step is recorded, so its C_x, C_y are always closed by the end-of-launch path; interleaved with
    shaken_run_alternate(1) on the same context."""
    seed = 600 + L
    J = np.linspace(0.4, 0.8, n_chains)
    q = np.linspace(0.7, 0.3, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    with shaken.Shaken(L, n_chains, seed, max_records=16) as s:
        s.init(0)
        for k in range(6):
            if k % 3 == 2:
                o.run_alternate(J, 1, 1)
                s.run_alternate(J, 1, 1)
            else:
                o.run_grid(J, q, 1, 1)
                s.run_grid(J, q, 1, 1)
        assert_same_state(s, o, f"L={L} chains={n_chains}")


# ----------------------------------------------------------------------------- coupled chains, coalescence
@pytest.mark.parametrize("packed,variant", [(False, 0), (False, 3), (True, 0)])
def test_coupled_chains_and_coalescence_times_match_oracle(packed, variant):
    """groups of chains that share their random numbers, sandwich start (top all +1, bottom all -1),
    coalescence time = first full step after which the sigma layers of a group agree.  Spins, records and the times
    must equal the oracle's bit for bit; the 32 x 32 torus is the paper's own size."""
    L, g, n_groups, seed, steps = 32, 2, 6, 13, 120
    J = np.repeat([0.2, 0.3, 0.44, 0.44, 0.6, 0.3], g)
    q = np.repeat([0.3, 1.0, 0.5, 2.0, 0.3, 0.1], g)
    o = so.Oracle(L, g * n_groups, seed)
    o.set_coupling(g)
    o.init(2)
    with shaken.Shaken(L, g * n_groups, seed, packed=packed, max_records=steps) as s:
        s.set_variant(variant)                         # 0: one CTA per group (kernel_small.cuh); 3: strip kernels + compare
        s.set_coupling(g)
        s.init(shaken.INIT_SANDWICH)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.get_spins(1), o.get_spins(1))
        for chunk in (1, 40, 79):                     # the times must not depend on how the run is split
            o.run_grid(J, q, chunk, 10)
            s.run_grid(J, q, chunk, 10)
            assert np.array_equal(s.coalescence(), o.coalescence()), chunk
        assert_same_state(s, o, f"coupled packed={packed}")
        coal = s.coalescence()
        assert coal.shape == (n_groups,) and np.any(coal > 0)
        sig = s.get_spins(0)
        for gi in range(n_groups):
            top, bot = sig[g * gi], sig[g * gi + 1]
            assert np.all(top >= bot)                  # ordering preserved
            assert (coal[gi] > 0) == bool(np.array_equal(top, bot))
        s.init(shaken.INIT_SANDWICH)
        assert np.all(s.coalescence() == -1)


def test_coupling_group_of_three_with_chain_offset_and_bookkeeping():
    L, g, seed = 48, 3, 5
    o_big = so.Oracle(L, 2 * g, seed)
    o_big.set_coupling(g)
    o_big.init(2)
    o_big.run(0.25, 0.4, 60, 0)
    with shaken.Shaken(L, g, seed) as s:               # second group alone: chains 3..5 of the batch
        s.set_chain_offset(g)
        s.set_coupling(g)
        s.init(shaken.INIT_SANDWICH)
        s.run(0.25, 0.4, 60, 0)
        assert np.array_equal(s.get_spins(0), o_big.get_spins(0)[g:])
        assert np.array_equal(s.coalescence(), o_big.coalescence()[1:])
        with pytest.raises(shaken.ShakenError):
            s.set_coupling(2)                          # must divide n_chains
        s.set_coupling(1)
        assert s.coalescence().size == 0


def test_propp_wilson_driver_draws_the_oracles_samples():
    """coupling from the past on the GPU (paper_1908_07341_b200/sampling.py) against the oracle's
    own driver (oracle/shaken_oracle.py: propp_wilson, pinned on the 3 x 3 torus): same look-back T, same samples."""
    from paper_1908_07341_b200 import sampling

    L, n_pairs, seed = 16, 24, 31
    qs = np.repeat(np.linspace(0.3, 1.5, n_pairs), 2)
    Js = np.repeat(np.linspace(0.15, 0.35, n_pairs), 2)
    o = so.Oracle(L, 2 * n_pairs, seed)
    o.set_coupling(2)
    want, T_want = so.propp_wilson(o, Js, qs, base=1 << 33)
    for packed in (False,):
        with shaken.Shaken(L, 2 * n_pairs, seed, packed=packed) as s:
            s.set_coupling(2)
            got, T = sampling.propp_wilson(s, Js, qs, base=1 << 33)
            assert T == T_want and np.array_equal(got, want)
            with pytest.raises(ValueError):
                sampling.propp_wilson(s, Js + np.tile([0.0, 0.1], n_pairs), qs)


@pytest.mark.parametrize("L,packed", [(32, False), (32, True), (176, False), (160, True)])
def test_diagonal_correlation_sums_match_oracle(L, packed):
    """SURVEY 8(f) rank 2 (Table 1: 32 x 32 box, l = 1, 2, 4, 8, 16): SW-NE and NW-SE sums of the
    sigma layer after a few steps, for distances that are and are not multiples of the word width, incl. l >= L."""
    n, seed = 3, 17
    ells = [0, 1, 2, 3, 4, 5, 8, 16, 31, 33, L - 1, L, L + 7]
    o = so.Oracle(L, n, seed)
    o.init(0)
    o.run_grid([0.3, 0.44, 0.6], [0.2, 1.0, 0.5], 5, 0)
    with shaken.Shaken(L, n, seed, packed=packed) as s:
        s.init(0)
        s.run_grid([0.3, 0.44, 0.6], [0.2, 1.0, 0.5], 5, 0)
        assert np.array_equal(s.diag_correlations(ells), o.diag_correlations(ells))
        with pytest.raises(shaken.ShakenError):
            s.diag_correlations([-1])


def test_batch_of_mid_size_chains_runs_in_the_one_cta_per_chain_path():
    """128 < L <= 288 with enough chains to fill the machine (the paper's (q,J) scan uses 200 x 200): one
    CTA per chain, whole run in one launch, rows of 13 vectors (not a power of two) walked by 512 threads."""
    L, n, seed = 208, 80, 3
    J = np.linspace(0.1, 0.9, n)
    q = np.linspace(2.0, 0.1, n)
    o = so.Oracle(L, n, seed)
    o.init(-1)                                         # the paper's scan starts from all -1
    o.run_grid(J, q, 5, 2)
    with shaken.Shaken(L, n, seed, max_records=4) as s:
        s.init(-1)
        l0 = s.launch_count
        s.run_grid(J, q, 3, 2)
        s.run_grid(J, q, 2, 2)
        assert s.launch_count - l0 == 2                # one launch per shaken_run call
        assert_same_state(s, o, "L=208 batch")
