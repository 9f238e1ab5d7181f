#!/usr/bin/env python
"""bench.py -- one JSON line for BASELINE.json's metric: spin site-updates/ns of the shaken-dynamics hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg1|cfg2|cfg3|cfg5|paper<L>] [--impl reference]

A *step* is one full shaken step over the whole workload: half-step 0 (eq. 15) and half-step 1 (eq. 16) of
every site of every chain, with the observable sums fused in as the workload prescribes.  Default workload:
BASELINE.json configs[3] ("cfg4": L=16384 int8, J=q=0.7, all +1, seed 3, six sums every step) -- the
configuration the metric is quoted on.

* ``value``     device-resident throughput: K steps timed with CUDA events on the stream the kernels run on.
* ``e2e``       the same job through the C ABI with HOST buffers inside the timed region: shaken_set_spins of sigma
                (the whole input: half-step 0 redraws every tau from sigma alone) from pinned host memory,
                shaken_run(K steps), shaken_observables and shaken_get_spins(sigma) back to the host.  Bytes per step
                are the totals divided by K.
* ``roofline``  dominant kernel (the half-step kernel, 2K launches in the timed region): algorithmic bytes per
                launch (2 B per site-update: read one source byte, write one target byte; 0.25 B bit-packed) over
                its mean duration, against the measured HBM copy bandwidth of MEASURED_PEAKS.json; nested: the integer
                multiplier view (``alu``) and the Philox-only ceiling measured in the same run through the library.
* ``workloads`` (default run only) the other four BASELINE.json workloads, a short timed leg each.
* ``cpu_baseline``  the oracle (oracle/, as it stands, single thread) timed on this box on a bounded sample.
* ``--impl reference``  for this tier the reference arm IS the oracle: times it on the host cores, each step a
                bounded band of rows of the same workload.

N > 1 (torchrun): the workload is replicated as independent chains, rank r simulating global chain r of an
N-chain batch (chains are independent units -- no data-path collective); ``--slabs`` shares ONE
lattice between the ranks instead (row slabs, one sigma row each way per step by peer stores: strong scaling).
SHAKEN_BENCH_ONE_DEVICE=1 (tests on a one-GPU box) lets all ranks of the replica arm use cuda:0, control plane over gloo.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "spin site-updates/ns"
UNIT = "site-updates/ns"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-workloads", action="store_true", help="skip the short legs on the other four BASELINE.json workloads")
    ap.add_argument("--slabs", action="store_true",
                    help="N ranks share ONE lattice of the named single-chain int8 workload as row slabs (strong scaling; one sigma "
                         "row each way per step by peer stores, DESIGN.md section 9) instead of running N replicas")
    ap.add_argument("--variant", type=int, default=0, choices=[0, 3, 8], help="code-path switch of shaken_set_variant (0 = automatic)")
    ap.add_argument("--cpu-multicore-leg", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--dynamics", default="shaken", choices=["shaken", "alternate"],
                    help="alternate: the even/odd heat bath on the square lattice (PAPER.md:276) on the same lattice, "
                         "chains, J and record cadence as the named workload; a step redraws every site once")
    return ap.parse_args()


def workload(name: str):
    from paper_1908_07341_b200 import workloads

    if name.startswith("paper"):        # the paper's own benchmark point at lattice side L: --workload paper2048
        return workloads.paper_benchmark_point(int(name[5:]))
    idx = {"cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}[name]
    return workloads.config(idx)


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ----------------------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.samples = []
        self._stop = threading.Event()
        self._th = None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [x.strip() for x in out.strip().splitlines()[0].split(",")]
                self.samples.append(parts)
            except Exception:
                pass
            self._stop.wait(0.05)

    def start(self):
        self._th = threading.Thread(target=self._run, daemon=True)
        self._th.start()

    def stop(self):
        self._stop.set()
        if self._th:
            self._th.join(timeout=10)

    def summary(self):
        if not self.samples:
            return None
        sm = sorted(float(s[0]) for s in self.samples if s[0].replace(".", "").isdigit())
        mx = [float(s[1]) for s in self.samples if s[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(s) > 3 + i and s[3 + i].lower().startswith("active") for s in self.samples)]
        pw = [float(s[2]) for s in self.samples if s[2].replace(".", "").isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "power_w_max": max(pw) if pw else None, "samples": len(self.samples)}


# ----------------------------------------------------------------------------------------- reference arm = oracle
def oracle_sample_step(w, src, band_rows, alternate=False):
    """One bounded 'step' of the oracle: both half-steps of `band_rows` rows of chain 0 of the workload."""
    from oracle import shaken_oracle as so

    if alternate:
        a = so.alt_half_step_rows(src, w.seed, 0, w.J[0], 0, 0, 0, band_rows)
        b = so.alt_half_step_rows(src, w.seed, 0, w.J[0], 0, 1, 0, band_rows)
        return a, b
    a = so.half_step_rows(src, w.seed, 0, w.J[0], w.q[0], 0, 0, 0, band_rows)
    b = so.half_step_rows(src, w.seed, 0, w.J[0], w.q[0], 0, 1, 0, band_rows)
    return a, b


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import shaken_oracle as so

    so.build()
    w = workload(args.workload)
    L = w.L
    band = max(1, min(L, (8 << 20) // L))                 # ~8 Mi sites per half-step
    src = np.ones((L, L), dtype=np.int8) if w.init == 1 else np.where(
        np.random.default_rng(w.seed).integers(0, 2, size=(L, L)) == 1, 1, -1).astype(np.int8)
    alt = args.dynamics == "alternate"
    per_step = (1 if alt else 2) * band * L                # alternate: each half-step redraws half the sites of the band
    for _ in range(max(args.warmup, 1)):
        oracle_sample_step(w, src, band, alt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample_step(w, src, band, alt)
    dt = time.perf_counter() - t0
    updates = float(per_step) * args.steps
    v = updates / (dt * 1e9)
    sample = f"{band} rows x {L} columns of one chain, both half-steps, per step ({per_step} site updates)"
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8", "data": "synthetic",
        "config": {"workload": w.name, "L": L, "n_chains": w.n_chains, "dynamics": args.dynamics,
                   "note": "oracle/shaken_oracle.c on host cores, bounded sample per step"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def cpu_baseline(w, alternate=False):
    """The oracle as it stands, single thread, about 10-30 s of work on the same workload shape."""
    from oracle import shaken_oracle as so

    so.build()
    L = w.L
    band = max(1, min(L, (256 << 20) // L))               # up to 256 Mi sites per half-step
    src = np.ones((L, L), dtype=np.int8)
    oracle_sample_step(w, src, min(band, 64), alternate)   # warm the code path
    t0 = time.perf_counter()
    reps = 0
    while True:                                            # whole half-step pairs until about 12 s of CPU work
        if alternate:
            so.alt_half_step_rows(src, w.seed, 0, w.J[0], reps, 0, 0, band)
            so.alt_half_step_rows(src, w.seed, 0, w.J[0], reps, 1, 0, band)
        else:
            so.half_step_rows(src, w.seed, 0, w.J[0], w.q[0], reps, 0, 0, band)
            so.half_step_rows(src, w.seed, 0, w.J[0], w.q[0], reps, 1, 0, band)
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= 12.0 or reps >= 64:
            break
    upd = (1.0 if alternate else 2.0) * band * L * reps
    return {"value": upd / (dt * 1e9), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{reps} x both half-steps of {band} rows x {L} columns of chain 0 ({int(upd)} site updates, {dt:.1f} s)",
            "host_cores_available": os.cpu_count()}


_MC = {}


def _mc_band(args):
    """Worker of cpu_baseline_multicore: one band of rows of one half-step by the oracle; returns a checksum only."""
    from oracle import shaken_oracle as so

    w_seed, J, q, t, half, r0, nrows, alternate = args
    src = _MC["src"]
    if alternate:
        out = so.alt_half_step_rows(src, w_seed, 0, J, t, half, r0, nrows)
    else:
        out = so.half_step_rows(src, w_seed, 0, J, q, t, half, r0, nrows)
    return int(out.sum(dtype=np.int64))


def cpu_baseline_multicore(w, alternate=False):
    """SURVEY 8(d), optional second line: the same oracle, unchanged, with the rows of a half-step split over all host
    cores by processes (legal because the randomness is a function of the site index).  About 5-10 s."""
    import multiprocessing as mp

    from oracle import shaken_oracle as so

    so.build()
    cores = os.cpu_count() or 1
    L = w.L
    band = max(cores, min(L, (256 << 20) // L))
    _MC["src"] = np.ones((L, L), dtype=np.int8)            # inherited by the forked workers, never pickled
    bounds = np.linspace(0, band, cores + 1).astype(int)
    with mp.get_context("fork").Pool(cores) as pool:
        def half(t, h):
            jobs = [(w.seed, w.J[0], w.q[0], t, h, int(bounds[i]), int(bounds[i + 1] - bounds[i]), alternate) for i in range(cores)]
            return pool.map(_mc_band, jobs)
        half(0, 0)                                         # warm the workers
        t0 = time.perf_counter()
        reps = 0
        while True:
            half(reps, 0)
            half(reps, 1)
            reps += 1
            dt = time.perf_counter() - t0
            if dt >= 5.0 or reps >= 64:
                break
    upd = (1.0 if alternate else 2.0) * band * L * reps
    return {"value": upd / (dt * 1e9), "unit": UNIT, "cores": cores, "kind": "oracle, rows split over processes",
            "sample": f"{reps} x both half-steps of {band} rows x {L} columns of chain 0 ({int(upd)} site updates, {dt:.1f} s)"}


# ----------------------------------------------------------------------------------------- our arm
def muls_per_site(w, alt):
    """IMAD.WIDE per site-update of the kernels this workload launches (17 or 18 per Philox4x32-10 call of 4 sites:
    rounds 0-1 hoisted; launches that carry the round-0 product by additions spend 17 -- philox.cuh)."""
    if alt:
        return 18 / 4.0                                    # kernel_alt.cuh: philox_site_words[_xn] without the carried product
    if w.packed:
        return 17 / 4.0                                    # kernel_pk.cuh: carried product in every launch
    if w.L <= 2048 and w.n_chains <= 148:
        return 18 / 4.0                                    # one-launch paths (kernel_small.cuh, kernel_band.cuh)
    if w.obs_every == 1:
        return 17 / 4.0                                    # kernel_i8.cuh: every launch carries sums, hence the product
    if w.obs_every == 0:
        return 18 / 4.0
    return (17.0 / w.obs_every + 18.0 * (1.0 - 1.0 / w.obs_every)) / 4.0


def time_workload(shaken, torch, dist, w, K, W, dev, stream, rank, world, alt, variant=0, before_timed=None, slabs=False):
    """W warm-up steps, then K steps timed with CUDA events on the library's stream.  Returns (context, ms, launches, run)."""
    if slabs:
        from paper_1908_07341_b200 import parallel

        s = parallel.open_slab(w.L, w.seed, world, rank, max_records=(K + W) // max(w.obs_every, 1) + 4 if w.obs_every else 0, stream=stream)
        parallel.connect_slabs_ipc(s)

        def run(n):
            s.run(w.J[0], w.q[0], n, w.obs_every)

        s.init(w.init)
        run(W)
        s.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)
        if before_timed:
            before_timed()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = s.launch_count
        e0.record(stream)
        run(K)
        e1.record(stream)
        e1.synchronize()
        torch.cuda.synchronize(dev)
        return s, e0.elapsed_time(e1), s.launch_count - l0, run
    s = shaken.Shaken(w.L, w.n_chains, w.seed, packed=w.packed, max_records=(K + W) // max(w.obs_every, 1) + 4 if w.obs_every else 1,
                      device=str(dev), stream=stream)
    s.set_chain_offset(rank * w.n_chains)
    if variant:
        s.set_variant(variant)
    J, q = w.J_array(), w.q_array()
    uniform = len(set(w.J)) == 1 and len(set(w.q)) == 1

    def run(n):
        if alt:
            s.run_alternate(w.J[0] if uniform else J, n, w.obs_every)
        elif uniform:
            s.run(w.J[0], w.q[0], n, w.obs_every)
        else:
            s.run_grid(J, q, n, w.obs_every)

    s.init(w.init)
    run(W)
    s.synchronize()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev)
    if before_timed:
        before_timed()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.launch_count
    e0.record(stream)
    run(K)
    e1.record(stream)
    e1.synchronize()
    torch.cuda.synchronize(dev)
    return s, e0.elapsed_time(e1), s.launch_count - l0, run


def rooflines(w, alt, ms, K, n_sms, sm_max_mhz, hbm_peak, philox_only, share=1.0):
    """HBM view (the metric's denominator), integer-multiplier view and the measured Philox-only ceiling of one workload."""
    bytes_per_update = 0.25 if w.packed else 2.0
    sites_per_launch = int(w.n_chains * w.L * w.L * share)   # share < 1: this rank's slab of a shared lattice
    if alt:
        bytes_per_update *= 2.0                            # in place on one array: read + write the array to redraw half of it
        sites_per_launch //= 2
    avg_launch_ms = ms / (2 * K)                           # two half-steps per step (a trailing bond-sum pass is inside ms)
    rate = sites_per_launch / (avg_launch_ms * 1e6)        # site-updates per ns of the half-step kernel
    mps = muls_per_site(w, alt)
    alu_peak = n_sms * 4 * 8 * sm_max_mhz * 1e6 / 1e9      # G IMAD.WIDE lane-operations per second
    return {"sites_per_launch": sites_per_launch, "avg_launch_us": avg_launch_ms * 1e3,
            "alg_bytes_per_launch": bytes_per_update * sites_per_launch,
            "hbm_achieved": bytes_per_update * rate, "hbm_frac": bytes_per_update * rate / hbm_peak,
            "alu_achieved": mps * rate, "alu_peak": alu_peak, "alu_frac": mps * rate / alu_peak, "muls_per_site": mps,
            "philox_frac": rate / philox_only if philox_only else None}


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_1908_07341_b200 import build as _build, shaken

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libshaken has no CPU fallback")
    if rank == 0:
        _build.build()
    # SHAKEN_BENCH_ONE_DEVICE=1 (tests on a one-GPU box): every rank uses device 0 and the control plane (barriers, the max
    # over ranks) runs over gloo -- NCCL refuses two ranks on one device.  Replica arm only: slabs wait for each other.
    one_dev = world > 1 and os.environ.get("SHAKEN_BENCH_ONE_DEVICE") == "1"
    if one_dev and args.slabs:
        raise SystemExit("bench.py: SHAKEN_BENCH_ONE_DEVICE is for the replica arm (the kernels of row slabs wait for each other)")
    dev_index = 0 if one_dev else local_rank
    torch.cuda.set_device(dev_index)
    dev = torch.device("cuda", dev_index)
    ctl = torch.device("cpu") if one_dev else dev           # where the tensors of the control-plane collectives live
    if world > 1:
        if one_dev:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=dev)
        dist.barrier()

    w = workload(args.workload)
    K, W = args.steps, max(args.warmup, 3)
    stream = torch.cuda.Stream(device=dev)
    n_local = w.n_chains                                   # weak scaling: every rank runs the whole named workload
    alt = args.dynamics == "alternate"
    uniform = len(set(w.J)) == 1 and len(set(w.q)) == 1

    sampler = ClockSampler(dev_index)
    slabs = bool(args.slabs)
    if slabs and (alt or w.packed or w.n_chains != 1):
        raise SystemExit("bench.py --slabs: needs a single-chain int8 workload of the shaken dynamics (cfg4, cfg2, paper<L>)")
    s, ms, launches, run = time_workload(shaken, torch, dist, w, K, W, dev, stream, rank, world, alt, args.variant,
                                         before_timed=sampler.start if rank == 0 else None, slabs=slabs)
    if world > 1:
        t = torch.tensor([ms], device=ctl, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    # nvidia-smi needs ~50 ms per sample: keep the same launch sequence running right after the timed region until at
    # least 1.5 s of load has been sampled (records are discarded; obs cadence unchanged).  Slabs of one lattice wait for
    # each other, so there every rank repeats the run the same number of times; replicas are independent (rank 0 only).
    reps = int(max(1.5 - ms * 1e-3, 0.0) / max(ms * 1e-3, 1e-6)) + 1
    if rank == 0 or (slabs and world > 1):
        for _ in range(reps):
            s.clear_records()
            run(K)
            s.synchronize()
    if rank == 0:
        sampler.stop()
    if world > 1:
        dist.barrier()

    updates_per_rank = (1.0 if alt else 2.0) * n_local * w.L * w.L * K   # alternate: a half-step redraws one colour
    if slabs:
        updates_per_rank /= world                          # strong scaling: the ranks share one lattice
    value = world * updates_per_rank / (ms * 1e6)

    # ------------------------------------------------------------------ e2e through the C ABI with host buffers
    e2e = None
    if not args.no_e2e and slabs:
        e2e = {"unavailable": "the e2e leg is measured on the replica arm (a slab holds a part of the lattice)"}
    elif not args.no_e2e:
        nsp = n_local * w.L * w.L
        h_sigma = torch.empty(nsp, dtype=torch.int8).pin_memory()
        h_out = torch.empty(nsp, dtype=torch.int8).pin_memory()
        n_rec = K // max(w.obs_every, 1) if w.obs_every else 0
        h_rec = torch.zeros(max(n_rec, 1) * n_local * 6, dtype=torch.int64).pin_memory()
        s.get_spins_into(0, h_sigma.data_ptr())
        s.clear_records()
        s.step = 0
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        # sigma is the whole input of a run: half-step 0 redraws every tau from sigma alone (eq. 15; SURVEY 8(c) reading 6,
        # "the dynamics never reads the initial tau"), and the alternate dynamics has no tau
        s.set_spins_from(0, h_sigma.data_ptr())
        run(K)
        got = s.observables_into(h_rec.data_ptr(), max(n_rec, 1))
        s.get_spins_into(0, h_out.data_ptr())
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], device=ctl, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": world * updates_per_rank / (dt * 1e9), "unit": UNIT,
               "h2d_bytes_per_step": nsp / K, "d2h_bytes_per_step": (nsp + got * n_local * 48) / K,
               "ms_total": dt * 1e3,
               "what": "shaken_set_spins(sigma) from pinned host + " + ("shaken_run_alternate(K)" if alt else "shaken_run(K)") +
                       " + shaken_observables + shaken_get_spins(sigma) to host; one upload and one download per run of K "
                       "steps (step k+1 reads the resident output of step k)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    s.close()

    # ------------------------------------------------------------------ rooflines of the half-step kernel
    # Top level: the HBM roofline BASELINE.json's metric names (2 B per site-update: read one source byte, write one
    # target byte; 0.25 B bit-packed) against the measured copy bandwidth.  Beside it what actually bounds the path
    # (DESIGN.md "Rooflines"): the integer multiplier -- 32 random bits per site cost 4.25-4.5 IMAD.WIDE, and a warp-wide
    # IMAD.WIDE holds an SMSP's 16-lane multiplier for 4 cycles (peak = n_SM x 4 SMSP x 8 lane-multiplies/clk x max SM
    # clock) -- and the rate of a Philox-only kernel measured in THIS run through the library (no memory traffic at all).
    hbm_peak, peak_src = measured_peak()
    props = torch.cuda.get_device_properties(dev)
    clk = sampler.summary() or {}
    sm_max_mhz = clk.get("sm_max_mhz") or 1965.0
    philox_only = None
    try:
        philox_only = shaken.philox_only_rate()
    except Exception as e:                                 # the hook must never cost the bench line
        philox_only = None
        print("bench.py: philox-only hook failed: %r" % (e,), file=sys.stderr)
    rl = rooflines(w, alt, ms, K, props.multi_processor_count, sm_max_mhz, hbm_peak, philox_only, 1.0 / world if slabs else 1.0)
    traffic, traffic_source = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic.txt")
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            traffic = tj.get(w.name + ("_alt" if alt else ""))
            traffic_source = tj.get("source")
        except Exception:
            traffic = None
    kernel = ("alt_half (packed)" if w.packed else "alt_strip_i8") if alt else ("half_step_pk" if w.packed else "half_step_i8")
    roofline = {"bound": "hbm", "achieved": rl["hbm_achieved"], "peak": hbm_peak, "unit": "GB/s", "frac": rl["hbm_frac"],
                "traffic": traffic,
                "traffic_source": traffic_source or "profiles/traffic.txt: dram__bytes_read.sum + dram__bytes_write.sum per launch "
                                                    "from the committed ncu --set full capture of this kernel (not measured in this run)",
                "peak_source": peak_src, "kernel": kernel,
                "algorithmic_bytes_per_launch": rl["alg_bytes_per_launch"], "avg_launch_us": rl["avg_launch_us"],
                "binding_resource": "integer pipes, not HBM: the ALU/dispatch port (83-85 % busy) ahead of the multiplier pipe (76 %); Philox4x32-10 at 32 random bits per site fills both (DESIGN.md Rooflines)",
                "alu": {"achieved": rl["alu_achieved"], "peak": rl["alu_peak"], "unit": "G IMAD.WIDE/s", "frac": rl["alu_frac"],
                        "imad_wide_per_site_update": rl["muls_per_site"],
                        "peak_source": "derived (DESIGN.md Rooflines): %d SMs x 4 SMSP x 8 wide multiplies/clk x %.0f MHz"
                                       % (props.multi_processor_count, sm_max_mhz),
                        "peak_site_updates_per_ns": rl["alu_peak"] / rl["muls_per_site"]},
                "philox_only_sites_per_ns": philox_only,
                "frac_of_philox_only": rl["philox_frac"],
                "philox_only_source": "measured in this run: shaken_selftest_philox_rate (the kernels' own Philox + one compare "
                                      "per word, no memory traffic), best of 3 launches, CUDA events"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong" if slabs else "weak", "vs_baseline": None,
        "dtype": "u32 bit-packed" if w.packed else "int8", "data": "synthetic",
        "config": {"workload": w.name, "dynamics": args.dynamics, "L": w.L, "n_chains_per_gpu": n_local, "J": w.J[0] if uniform else "grid",
                   "q": (w.q[0] if uniform else "grid") if not alt else None, "obs_every": w.obs_every, "init": w.init, "seed": w.seed,
                   "l2": "inputs larger than L2 (2 x %.0f MB per step)" % (shaken_bytes(w) / 1e6) if shaken_bytes(w) > 126e6
                         else "working set fits L2 (launch/latency-bound regime)",
                   "parallelism": ("row slabs of one lattice, one sigma row each way per step by peer stores" if slabs else
                                   "replicas (independent chains, no collective)") if world > 1 or slabs else "single GPU"},
        "clocks": sampler.summary(),
        "e2e": e2e,
        "gpu_launches": int(launches),
        "roofline": roofline,
    }

    # ------------------------------------------------------------------ the other workloads of BASELINE.json (north_star:
    # "report throughput on the five synthetic workloads"), a few hundred ms each, same timing method
    if world == 1 and not args.no_workloads and args.workload == "cfg4" and not alt:
        others = {}
        for name, k in (("cfg1", 2000), ("cfg2", 2000), ("cfg3", 60), ("cfg5", 40)):
            try:
                wo = workload(name)
                so_, ms_o, launches_o, _ = time_workload(shaken, torch, dist, wo, k, 5, dev, stream, 0, 1, False, 0)
                so_.close()
                r = rooflines(wo, False, ms_o, k, props.multi_processor_count, sm_max_mhz, hbm_peak, philox_only)
                others[name] = {"value": 2.0 * wo.n_chains * wo.L * wo.L * k / (ms_o * 1e6), "unit": UNIT, "steps": k,
                                "ms_per_step": ms_o / k, "us_per_step": 1e3 * ms_o / k, "launches": int(launches_o),
                                "hbm_frac": r["hbm_frac"], "alu_frac": r["alu_frac"], "frac_of_philox_only": r["philox_frac"],
                                "layout": "u32 bit-packed" if wo.packed else "int8", "L": wo.L, "n_chains": wo.n_chains,
                                "obs_every": wo.obs_every}
                del so_
                torch.cuda.empty_cache()
            except Exception as e:
                others[name] = {"unavailable": repr(e)[:200]}
        others[w.name] = {"value": value, "unit": UNIT, "steps": K, "ms_per_step": ms / K, "us_per_step": 1e3 * ms / K,
                          "launches": int(launches), "hbm_frac": rl["hbm_frac"], "alu_frac": rl["alu_frac"],
                          "frac_of_philox_only": rl["philox_frac"], "layout": "int8", "L": w.L, "n_chains": w.n_chains,
                          "obs_every": w.obs_every}
        line["workloads"] = others

    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(w, alt)
        try:
            # in a fresh interpreter (this one holds a CUDA context and must not be forked), bounded in time
            out = subprocess.run([sys.executable, os.path.abspath(__file__), "--cpu-multicore-leg", "--workload", args.workload,
                                  "--dynamics", args.dynamics], capture_output=True, text=True, timeout=240).stdout
            line["cpu_baseline_multicore"] = json.loads(out.strip().splitlines()[-1])
        except Exception as e:                             # never let the optional leg cost the bench line
            line["cpu_baseline_multicore"] = {"unavailable": repr(e)[:200]}
    elif world > 1:
        line["cpu_baseline"] = None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def shaken_bytes(w):
    n = w.n_chains * w.L * w.L
    return n / 8 if w.packed else n


def main():
    args = parse_args()
    if args.cpu_multicore_leg:
        print(json.dumps(cpu_baseline_multicore(workload(args.workload), args.dynamics == "alternate")))
        return 0
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
