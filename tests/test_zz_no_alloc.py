"""``-m gpu``: shaken_run_static (include/shaken.h), the entry point that allocates nothing -- the band kernels with their
hand-over scratch in a file-scope device array -- against the existing context path (shaken_run on an int8 context, itself
compared with the oracle bit for bit elsewhere) and, on one small lattice, against the oracle directly.  Integer work:
the comparison is bit-exact, as in every parity test here.  Every case makes TWO calls in a row on the same buffers (the
static array keeps the first call's contents; the second call must clear what it uses and continue at t0 = n1).

Collected last on purpose (the file name): the suite runs with ``pytest -x``."""
import numpy as np
import pytest

from paper_1908_07341_b200 import shaken

pytestmark = pytest.mark.gpu


def _two_calls(L, n_chains, seed, J, q, n1, n2, obs, init=0):
    import torch

    dev = torch.device("cuda", 0)
    n_rec = (n1 + n2) // max(obs, 1) + 2 if obs else 0
    with shaken.Shaken(L, n_chains, seed, max_records=max(n_rec, 1)) as ref:
        ref.init(init)
        sigma = torch.from_numpy(ref.get_spins(0).copy()).to(dev)
        tau = torch.full_like(sigma, 0x55)                       # never read: half-step 0 redraws all of tau
        rec = torch.full((max(n_rec, 1), n_chains, 6), 77, dtype=torch.int64, device=dev)   # garbage: the call zeroes what it fills
        stream = torch.cuda.current_stream(dev)
        torch.cuda.synchronize(dev)
        shaken.static_setup()
        t0, done = 0, 0
        for k, n in enumerate((n1, n2)):
            free_before = torch.cuda.mem_get_info(dev)[0]
            shaken.run_static(sigma.data_ptr(), tau.data_ptr(), L, n_chains, seed, t0, J, q, n, obs,
                              rec.data_ptr() if obs else 0, rec.shape[0] if obs else 0, stream.cuda_stream)
            torch.cuda.synchronize(dev)
            free_after = torch.cuda.mem_get_info(dev)[0]
            if k == 1:                                           # (the first launch of a kernel may load its module)
                assert free_after == free_before, "the second call changed the amount of free device memory"
            ref.run(J, q, n, obs)
            what = f"L={L} chains={n_chains} call {k + 1}"
            assert np.array_equal(sigma.cpu().numpy(), ref.get_spins(0)), "sigma differs, " + what
            assert np.array_equal(tau.cpu().numpy(), ref.get_spins(1)), "tau differs, " + what
            want = ref.observables()[done:]
            if obs:
                got = rec.cpu().numpy()
                assert np.array_equal(got[: len(want)], want), "records differ, " + what
                assert np.all(got[len(want):] == 77), "slots beyond the run's records were touched, " + what
                rec.fill_(77)
            else:
                assert len(want) == 0
            done += len(want)
            t0 += n
        return sigma.cpu().numpy(), tau.cpu().numpy()


@pytest.mark.parametrize("L,n_chains,n1,n2,obs", [
    (1024, 1, 7, 6, 2),      # cfg 2's shape: bands of seven rows, the data-flow kernel; second call starts inside a record interval
    (2048, 1, 3, 4, 1),      # the largest lattice: bands of 14 rows, the two-phase kernel, 2.4 MB of the 2.5 MiB scratch
    (272, 3, 9, 5, 3),       # several chains, ragged rows (17 vectors)
    (1024, 4, 3, 2, 0),      # four chains, tall bands, no records (rec = NULL)
])
def test_static_entry_point_matches_the_context_path_on_two_calls_in_a_row(L, n_chains, n1, n2, obs):
    _two_calls(L, n_chains, 20 + L + n_chains, 0.6585, 0.6585, n1, n2, obs)


def test_static_entry_point_matches_the_oracle():
    from oracle import shaken_oracle as so

    L, seed, J, q = 144, 5, 0.5, 0.8
    sigma, tau = _two_calls(L, 1, seed, J, q, 4, 3, 1)
    o = so.Oracle(L, 1, seed)
    o.init(0)
    o.run(J, q, 7, 1)
    assert np.array_equal(sigma, o.get_spins(0)) and np.array_equal(tau, o.get_spins(1))
    o.close()


def test_static_entry_point_rejects_what_does_not_fit():
    import torch

    buf = torch.zeros(4096 * 4096, dtype=torch.int8, device="cuda:0")
    p = buf.data_ptr()
    for L, n in [(4096, 1), (128, 1), (1000, 1), (2048, 4), (1024, 1000)]:
        with pytest.raises(shaken.ShakenError) as e:
            shaken.run_static(p, p, L, n, 1, 0, 0.5, 0.5, 1)
        assert e.value.code == shaken.EINVAL, (L, n, str(e.value))
    with pytest.raises(shaken.ShakenError) as e:
        shaken.run_static(p, p, 2048, 4, 1, 0, 0.5, 0.5, 1)
    assert "maximum" in str(e.value)
    with pytest.raises(shaken.ShakenError) as e:                 # three records, room for two
        shaken.run_static(p, p + 1024 * 1024, 1024, 1, 1, 0, 0.5, 0.5, 3, 1, p + 2 * 1024 * 1024, 2)
    assert e.value.code == shaken.ENOSPC
    with pytest.raises(shaken.ShakenError):                      # misaligned
        shaken.run_static(p + 4, p, 1024, 1, 1, 0, 0.5, 0.5, 1)
    shaken.run_static(p, p, 1024, 1, 1, 0, 0.5, 0.5, 0)          # zero steps: nothing to do, no launch
    torch.cuda.synchronize()
