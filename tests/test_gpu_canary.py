"""Out-of-bounds WRITE check (``-m gpu``).  compute-sanitizer is closed on this GPU pool, so this is the
poor man's memcheck: sigma, tau and the record buffer are carved out of larger torch tensors filled with a canary pattern,
bound through shaken_bind, every kernel family is run over ragged shapes, and the canaries before and after each buffer
must be untouched (and the results still equal the oracle's, so the kernels did use the buffers they were given)."""
import numpy as np
import pytest

from oracle import shaken_oracle as so
from paper_1908_07341_b200 import shaken

pytestmark = pytest.mark.gpu

GUARD = 1 << 16          # bytes of canary on either side (multiple of 16)


def carve(torch, nbytes, dtype_bytes=1):
    raw = torch.full((GUARD + nbytes + GUARD,), 0x5A, dtype=torch.uint8, device="cuda:0")
    return raw, raw[GUARD:GUARD + nbytes]


@pytest.mark.parametrize("L,n_chains,packed,variant,alt", [
    (16, 3, False, 0, False), (48, 2, False, 0, False), (64, 1, False, 0, False),      # one-SM kernel, cluster kernel
    (272, 3, False, 0, False), (528, 1, False, 0, False), (304, 37, False, 0, False),  # band kernel (ragged bands)
    (528, 1, False, 3, False), (144, 5, False, 8, False), (1040, 2, False, 3, False),  # strip kernels: block tasks, per-warp ranges
    (544, 2, True, 0, False), (64, 3, True, 0, False),                                # packed
    (272, 2, False, 0, True), (528, 1, False, 3, True), (64, 2, False, 0, True), (544, 2, True, 0, True)])   # alternate dynamics
def test_no_kernel_writes_outside_its_buffers(L, n_chains, packed, variant, alt):
    import torch

    seed, steps = 77 + L, 5
    J = np.linspace(0.3, 0.7, n_chains)
    q = np.linspace(0.9, 0.4, n_chains)
    o = so.Oracle(L, n_chains, seed)
    o.init(0)
    if alt:
        o.run_alternate(J, steps, 2)
    else:
        o.run_grid(J, q, steps, 2)
    with shaken.Shaken(L, n_chains, seed, packed=packed, use_torch=False) as s:
        nb = int(s._lib.shaken_spin_bytes(s._h))
        raw_s, sig = carve(torch, nb)
        raw_t, tau = carve(torch, nb)
        rec_bytes = 4 * n_chains * 6 * 8
        raw_r, rec = carve(torch, rec_bytes)
        stream = torch.cuda.current_stream()
        s._ck(s._lib.shaken_bind(s._h, sig.data_ptr(), tau.data_ptr(), rec.data_ptr(), rec_bytes, stream.cuda_stream))
        s._tensors = (raw_s, raw_t, raw_r, stream)          # keep them alive
        s.set_variant(variant)
        s.init(0)
        if alt:
            s.run_alternate(J, 3, 2)
            s.run_alternate(J, steps - 3, 2)
        else:
            s.run_grid(J, q, 3, 2)
            s.run_grid(J, q, steps - 3, 2)
        assert np.array_equal(s.get_spins(0), o.get_spins(0)) and np.array_equal(s.observables(), o.observables())
        torch.cuda.synchronize()
        for name, raw, n in (("sigma", raw_s, nb), ("tau", raw_t, nb), ("records", raw_r, rec_bytes)):
            assert bool((raw[:GUARD] == 0x5A).all()), f"write below the {name} buffer"
            assert bool((raw[GUARD + n:] == 0x5A).all()), f"write above the {name} buffer"
