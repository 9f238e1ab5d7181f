"""Parity (``-m gpu``) of row-slab sharding (second bullet; include/shaken.h shaken_create_slab): ONE lattice
split into slabs of rows, every slab its own libshaken context, the slabs exchanging one sigma row each way per full
step through their inboxes.  Only one GPU is available, so the slabs live on the same device and are advanced ONE AFTER
THE OTHER on the same stream (all publish, then each runs a step): no kernel ever waits for a kernel that has not been
launched.  The kernels, the halo logic, the stamps and the per-slab records are exactly those of a multi-GPU run; only
the transport (peer stores over NVLink, IPC handles) is not exercised.  Expected values: the oracle's unsplit lattice."""
import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import parallel, shaken

pytestmark = pytest.mark.gpu


def open_ring(L, seed, bounds, max_records):
    slabs = [shaken.ShakenSlab(L, r0, r1 - r0, seed, max_records=max_records) for r0, r1 in zip(bounds[:-1], bounds[1:])]
    n = len(slabs)
    for k, s in enumerate(slabs):
        s.connect(slabs[(k - 1) % n].inbox(), slabs[(k + 1) % n].inbox())
    return slabs


@pytest.mark.parametrize("L,bounds", [(64, [0, 64]), (64, [0, 32, 64]), (272, [0, 100, 102, 272]), (528, [0, 176, 352, 528]),
                                      (1056, [0, 2, 530, 1056])])
def test_slabs_of_one_lattice_match_the_unsplit_oracle(L, bounds):
    seed, steps, J, q = 7 + L, 7, 0.55, 0.8
    o = so.Oracle(L, 1, seed)
    o.init(0)
    o.run(J, q, steps, 2)
    slabs = open_ring(L, seed, bounds, steps)
    try:
        for s in slabs:
            s.init(0)
        for t in range(steps):
            for s in slabs:
                s.exchange()                      # all slabs publish before any of them waits
            for s in slabs:
                s.run(J, q, 1, 2)
        sigma = np.vstack([s.get_spins(0) for s in slabs])
        tau = np.vstack([s.get_spins(1) for s in slabs])
        assert np.array_equal(sigma, o.get_spins(0)[0]), "sigma differs"
        assert np.array_equal(tau, o.get_spins(1)[0]), "tau differs"
        rec = sum(s.observables() for s in slabs)
        assert np.array_equal(rec, o.observables()), "summed records differ"
        assert all(s.step == steps for s in slabs)
    finally:
        for s in slabs:
            s.close()


@pytest.mark.parametrize("k", range(16))
def test_random_slab_splits_match_the_unsplit_oracle(k):
    """Seeded random splits (1-5 slabs of at least two rows, any boundaries), sizes, starts, couplings, step counters and
    record intervals; several steps per driver round where a single slab is its own neighbour."""
    rng = np.random.default_rng(5100 + k)
    L = int(rng.choice([32, 64, 144, 272, 400, 528, 1040]))
    n_slabs = int(rng.integers(1, 6))
    while True:
        cuts = sorted(int(c) for c in rng.choice(np.arange(2, L - 1), size=n_slabs - 1, replace=False)) if n_slabs > 1 else []
        bounds = [0] + cuts + [L]
        if all(b - a >= 2 for a, b in zip(bounds[:-1], bounds[1:])):
            break
    seed, init = int(rng.integers(0, 2**62)), int(rng.choice([0, 0, 1, -1]))
    J, q = float(rng.choice([0.0, 0.3, 0.6585, 0.9])), float(rng.choice([0.0, 0.4, 0.6585, 10.0]))
    steps, obs = int(rng.integers(2, 9)), int(rng.choice([0, 1, 2, 3]))
    t0 = int(rng.choice([0, 5, (1 << 32) - 2, (1 << 41) + 1]))
    o = so.Oracle(L, 1, seed)
    o.init(init)
    o.step = t0
    o.run(J, q, steps, obs)
    slabs = open_ring(L, seed, bounds, steps + 1)
    try:
        for s in slabs:
            s.init(init)
            s.step = t0
        for t in range(steps):
            for s in slabs:
                s.exchange()
            for s in slabs:
                s.run(J, q, 1, obs)
        what = f"L={L} bounds={bounds} steps={steps} obs={obs} t0={t0}"
        assert np.array_equal(np.vstack([s.get_spins(0) for s in slabs]), o.get_spins(0)[0]), "sigma differs " + what
        assert np.array_equal(np.vstack([s.get_spins(1) for s in slabs]), o.get_spins(1)[0]), "tau differs " + what
        want = o.observables()
        if len(want):
            assert np.array_equal(sum(s.observables() for s in slabs), want), "summed records differ " + what
        else:
            assert all(len(s.observables()) == 0 for s in slabs)
    finally:
        for s in slabs:
            s.close()


def test_single_slab_runs_many_steps_per_call_and_resumes():
    """One slab covering the whole lattice is its own neighbour: shaken_run(n) then needs no driver in between (each step
    publishes to itself), records every step, run split in two calls, set_spins in between."""
    L, seed, J, q = 528, 99, 0.7, 0.3
    o = so.Oracle(L, 1, seed)
    o.init(1)
    o.run(J, q, 9, 1)
    s = shaken.ShakenSlab(L, 0, L, seed, max_records=16)
    try:
        ptr = s.inbox()
        s.connect(ptr, ptr)
        s.init(1)
        s.run(J, q, 4, 1)
        mid = s.get_spins(0).copy()
        s.set_spins(0, mid)                       # forgets the published rows: the next run publishes again
        s.run(J, q, 5, 1)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)[0]) and np.array_equal(s.get_spins(1), o.get_spins(1)[0])
        assert np.array_equal(s.observables(), o.observables())
    finally:
        s.close()


def test_slab_argument_and_state_errors():
    lib = shaken.lib()
    with pytest.raises(shaken.ShakenError):
        shaken.ShakenSlab(64, 0, 1, 1)            # fewer than two rows
    with pytest.raises(shaken.ShakenError):
        shaken.ShakenSlab(64, 60, 8, 1)           # beyond the lattice
    s = shaken.ShakenSlab(64, 0, 32, 1)
    try:
        s.init(1)
        with pytest.raises(shaken.ShakenError) as e:
            s.run(0.5, 0.5, 1, 0)                 # not connected
        assert e.value.code == shaken.ESTATE
        with pytest.raises(shaken.ShakenError):
            s.run_alternate(0.4, 1, 0)
        assert parallel.slab_shard(64, 2, 1) == (32, 32)
    finally:
        s.close()


def _device_count():
    try:
        import torch

        return torch.cuda.device_count()
    except Exception:
        return 0


@pytest.mark.skipif(_device_count() < 2, reason="needs two GPUs (the N > 1 arm of bench.py under torchrun)")
@pytest.mark.parametrize("extra", [[], ["--slabs"]])
def test_bench_two_ranks_under_torchrun(extra):
    """The N > 1 arm of bench.py exactly as the driver launches it: replicas (weak scaling, no collective) and row slabs
    of one lattice (strong scaling, peer stores through CUDA IPC inboxes)."""
    import json
    import os
    import socket
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3",
           "--no-cpu-baseline", "--workload", "paper4096"] + extra
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["value"] > 0
    assert line["scaling"] == ("strong" if extra else "weak")


def test_bench_replica_arm_with_two_ranks_on_one_device():
    """The N > 1 replica arm of bench.py (rank -> chain offset, barriers, max over ranks, rank 0 prints, the others exit 0)
    under torchrun with two ranks that share cuda:0 (SHAKEN_BENCH_ONE_DEVICE=1: control plane over gloo, since NCCL refuses
    two ranks on one device).  The replicas are independent -- no kernel of one rank waits for the other -- so this is safe
    on one GPU; the value it prints is not a measurement.  The NCCL plumbing itself needs two devices (test above)."""
    import json
    import os
    import socket
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3",
           "--no-cpu-baseline", "--no-workloads", "--workload", "paper4096"]
    env = dict(os.environ, SHAKEN_BENCH_ONE_DEVICE="1")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, "rank 0 alone prints the line"
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["value"] > 0 and line["scaling"] == "weak"
    assert line["e2e"]["value"] > 0 and line["gpu_launches"] >= 6


def _ipc_worker(rank, world, L, seed, steps, J, q, barrier, handles, results):
    """One slab per PROCESS, both on cuda:0, inboxes connected through CUDA IPC handles.  Host barriers around every step
    make sure a rank's rows are published (and the stream drained) before the other rank's kernels look for them, so no
    kernel ever waits for a kernel of the other process; what is exercised is the IPC mapping and the peer stores."""
    import numpy as np
    import torch

    from paper_1908_07341_b200 import parallel, shaken

    torch.cuda.set_device(0)
    s = parallel.open_slab(L, seed, world, rank, max_records=steps)
    try:
        handles[rank] = s.ipc_export()
        barrier.wait()
        below, above = parallel.slab_neighbours(world, rank)
        s.ipc_connect(bytes(handles[below]), bytes(handles[above]))
        s.init(0)
        for _ in range(steps):
            s.exchange()
            s.synchronize()
            barrier.wait()
            s.run(J, q, 1, 1)
            s.synchronize()
            barrier.wait()
        s.exchange()
        s.synchronize()
        barrier.wait()
        results[rank] = (s.get_spins(0).copy(), s.observables().copy())
        barrier.wait()                                   # nobody unmaps while the neighbour may still be reading
    finally:
        s.close()


def test_two_processes_exchange_slab_rows_through_cuda_ipc():
    import torch.multiprocessing as mp

    L, seed, steps, J, q = 272, 31, 4, 0.6, 0.5
    ctx = mp.get_context("spawn")
    mgr = ctx.Manager()
    handles, results = mgr.dict(), mgr.dict()
    barrier = ctx.Barrier(2)
    procs = [ctx.Process(target=_ipc_worker, args=(r, 2, L, seed, steps, J, q, barrier, handles, results)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=180)
    alive = [p for p in procs if p.is_alive()]
    for p in alive:
        p.kill()
    assert not alive, "a slab process did not finish"
    assert all(p.exitcode == 0 for p in procs), [p.exitcode for p in procs]
    o = so.Oracle(L, 1, seed)
    o.init(0)
    o.run(J, q, steps, 1)
    sigma = np.vstack([results[0][0], results[1][0]])
    assert np.array_equal(sigma, o.get_spins(0)[0]), "sigma differs"
    assert np.array_equal(results[0][1] + results[1][1], o.observables()), "summed records differ"
