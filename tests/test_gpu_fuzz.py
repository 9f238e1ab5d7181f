"""Randomised parity (``-m gpu``): seeded random jobs -- lattice size, layout, number of chains, coupling groups, start,
couplings (uniform or per chain), code-path switch, step counter, and a sequence of calls of both dynamics with random
lengths and record intervals -- run through the C ABI and through the CPU oracle; spins, records, coalescence times and
the step counter must agree bit for bit after every call.  The hand-picked cases of test_gpu_parity.py /
test_gpu_alternate.py aim at known edges; this one looks for the combinations nobody thought of.  Sizes keep the
oracle's share at a few tenths of a second per job (eq. 14-16 :157-172 and reading 20 of DESIGN.md are what
both sides implement; nothing here is specific to one kernel)."""
import os

import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import shaken

pytestmark = pytest.mark.gpu

N_JOBS = int(os.environ.get("SHAKEN_FUZZ_JOBS", "64"))      # a longer hunt: SHAKEN_FUZZ_JOBS=1000 python -m pytest tests/test_gpu_fuzz.py -m gpu


def _job(k: int):
    rng = np.random.default_rng(77_000 + k)
    packed = bool(rng.integers(0, 4) == 0)
    unit = 32 if packed else 16
    # sizes: around the switches between the one-SM, cluster, band and strip kernels, ragged rows, one-vector rows
    Ls = [unit, 2 * unit, 3 * unit, 64, 96, 128, 144, 160, 208, 256, 272, 288, 304, 320, 352, 416, 512, 528, 544]
    L = int(rng.choice([x for x in Ls if x % unit == 0]))
    group = int(rng.choice([1, 1, 1, 2, 3]))
    n_groups = int(rng.integers(1, 5 if L <= 160 else 3))
    n_chains = group * n_groups
    variant = int(rng.choice([0, 0, 0, 3, 8])) if not packed else int(rng.choice([0, 3]))
    init = int(rng.choice([shaken.INIT_SANDWICH, shaken.INIT_SANDWICH, shaken.INIT_IID])) if group > 1 else int(rng.choice([1, -1, 0, 0]))
    t0 = int(rng.choice([0, 0, 1, 7, (1 << 31) - 3, (1 << 32) - 1, (1 << 40) + 5]))
    chain0 = int(rng.choice([0, 0, 3, 1000]))
    per_chain = bool(rng.integers(0, 2)) or group > 1
    Jg = rng.choice([0.0, 0.2, 0.44, 0.6585, 0.9, -0.3], size=n_groups)
    qg = rng.choice([0.0, 0.1, 0.5, 0.6585, 2.0, 10.0], size=n_groups)
    J, q = np.repeat(Jg, group), np.repeat(qg, group)            # members of a group share their couplings
    budget = int(1.5e7 / (2 * n_chains * L * L)) + 2               # full steps the oracle does in about a quarter of a second
    calls = []
    for _ in range(int(rng.integers(1, 5))):
        n = int(rng.integers(1, max(2, min(budget, 40))))
        obs = int(rng.choice([0, 1, 1, 2, 3, 7]))
        alt = bool(rng.integers(0, 4) == 0)                      # the alternate heat bath on sigma (L is even)
        calls.append((alt, n, obs))
    return dict(L=L, packed=packed, group=group, n_chains=n_chains, variant=variant, init=init, t0=t0, chain0=chain0,
                per_chain=per_chain, J=J, q=q, calls=calls, seed=int(rng.integers(0, 2**62)))


@pytest.mark.parametrize("k", range(N_JOBS))
def test_random_job_matches_oracle(k):
    j = _job(k)
    L, n_chains = j["L"], j["n_chains"]
    max_rec = sum(n for _, n, _ in j["calls"]) + 4
    # the oracle has no chain offset: chain c of the library's context is chain chain0 + c of a larger oracle batch
    # when groups are not split (chain0 a multiple of the group size), so run that batch's tail only where it is cheap
    chain0 = j["chain0"] if j["chain0"] % j["group"] == 0 and j["chain0"] <= 3 else 0
    o = so.Oracle(L, chain0 + n_chains, j["seed"])
    J_o = np.concatenate([np.full(chain0, 0.1), j["J"]])
    q_o = np.concatenate([np.full(chain0, 0.1), j["q"]])
    with shaken.Shaken(L, n_chains, j["seed"], packed=j["packed"], max_records=max_rec) as s:
        s.set_variant(j["variant"])
        if chain0:
            s.set_chain_offset(chain0)
        if j["group"] > 1:
            s.set_coupling(j["group"])
            o.set_coupling(j["group"])
        s.init(j["init"])
        o.init(j["init"])
        s.step = j["t0"]
        o.step = j["t0"]
        what = f"job {k}: {j}"
        for alt, n, obs in j["calls"]:
            if alt:
                Ja = np.abs(j["J"]) if j["per_chain"] else float(abs(j["J"][0]))
                s.run_alternate(Ja, n, obs)
                o.run_alternate(np.concatenate([np.full(chain0, 0.1), np.broadcast_to(Ja, (n_chains,))]), n, obs)
            elif j["per_chain"]:
                s.run_grid(j["J"], j["q"], n, obs)
                o.run_grid(J_o, q_o, n, obs)
            else:
                s.run(j["J"][0], j["q"][0], n, obs)
                o.run_grid(np.concatenate([np.full(chain0, 0.1), np.full(n_chains, j["J"][0])]),
                           np.concatenate([np.full(chain0, 0.1), np.full(n_chains, j["q"][0])]), n, obs)
            assert s.step == o.step, what
            assert np.array_equal(s.get_spins(0), o.get_spins(0)[chain0:]), f"sigma differs, {what}"
            assert np.array_equal(s.get_spins(1), o.get_spins(1)[chain0:]), f"tau differs, {what}"   # (untouched by the alternate dynamics)
            assert np.array_equal(s.observables(), o.observables()[:, chain0:]), f"records differ, {what}"
            if j["group"] > 1:
                assert np.array_equal(s.coalescence(), o.coalescence()[chain0 // j["group"]:]), f"coalescence differs, {what}"
    o.close()
