"""Thin Python binding of libshaken (include/shaken.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of ``csrc/``; this module loads ``libshaken.so`` with
ctypes and passes plain pointers and sizes.  PyTorch is used only to own device memory and the stream
(``Shaken(..., use_torch=True)`` borrows two int8/int32 tensors and an int64 record tensor through
``shaken_bind``); without torch the library allocates with cudaMalloc itself.

There is no CPU fallback: if the shared library has not been built, importing :func:`lib` raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libshaken.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENOSPC = 0, -1, -2, -3, -4, -5
INT8, PACKED = 0, 1
INIT_UP, INIT_DOWN, INIT_IID, INIT_SANDWICH = 1, -1, 0, 2
N_OBS = 6
OBS_NAMES = ("M_sigma", "M_tau", "E_J", "E_q", "C_x", "C_y")

# every symbol include/shaken.h declares: (name, restype, argtypes)
_p = C.c_void_p
SIGNATURES = {
    "shaken_create": (C.c_int, [C.POINTER(_p), C.c_int32, C.c_int32, C.c_uint64, C.c_uint32]),
    "shaken_destroy": (C.c_int, [_p]),
    "shaken_spin_bytes": (C.c_size_t, [_p]),
    "shaken_record_bytes": (C.c_size_t, [_p]),
    "shaken_bind": (C.c_int, [_p, _p, _p, _p, C.c_size_t, _p]),
    "shaken_reserve_records": (C.c_int, [_p, C.c_int64]),
    "shaken_init": (C.c_int, [_p, C.c_int]),
    "shaken_run": (C.c_int, [_p, C.c_double, C.c_double, C.c_int64, C.c_int64]),
    "shaken_run_grid": (C.c_int, [_p, _p, _p, C.c_int64, C.c_int64]),
    "shaken_alt_thresholds": (C.c_int, [C.c_double, C.POINTER(C.c_uint32)]),
    "shaken_run_alternate": (C.c_int, [_p, C.c_double, C.c_int64, C.c_int64]),
    "shaken_run_alternate_grid": (C.c_int, [_p, _p, C.c_int64, C.c_int64]),
    "shaken_observables": (C.c_int64, [_p, _p, C.c_int64]),
    "shaken_num_records": (C.c_int64, [_p]),
    "shaken_clear_records": (C.c_int, [_p]),
    "shaken_get_spins": (C.c_int, [_p, C.c_int, _p]),
    "shaken_set_spins": (C.c_int, [_p, C.c_int, _p]),
    "shaken_get_step": (C.c_int, [_p, C.POINTER(C.c_uint64)]),
    "shaken_set_step": (C.c_int, [_p, C.c_uint64]),
    "shaken_set_chain_offset": (C.c_int, [_p, C.c_uint32]),
    "shaken_set_coupling": (C.c_int, [_p, C.c_int32]),
    "shaken_coalescence": (C.c_int64, [_p, _p, C.c_int64]),
    "shaken_diag_correlations": (C.c_int, [_p, _p, C.c_int32, _p]),
    "shaken_synchronize": (C.c_int, [_p]),
    "shaken_thresholds": (C.c_int, [C.c_double, C.c_double, C.POINTER(C.c_uint32)]),
    "shaken_philox_words": (C.c_int, [_p, _p, _p, C.c_int64]),
    "shaken_launch_count": (C.c_int64, [_p]),
    "shaken_set_variant": (C.c_int, [_p, C.c_int]),
    "shaken_adopt_spins": (C.c_int, [_p]),
    "shaken_create_slab": (C.c_int, [C.POINTER(_p), C.c_int32, C.c_int32, C.c_int32, C.c_uint64]),
    "shaken_set_stream": (C.c_int, [_p, _p]),
    "shaken_slab_inbox": (C.c_int, [_p, C.POINTER(_p), C.POINTER(C.c_size_t)]),
    "shaken_slab_connect": (C.c_int, [_p, _p, _p]),
    "shaken_slab_ipc_export": (C.c_int, [_p, _p]),
    "shaken_slab_ipc_connect": (C.c_int, [_p, _p, _p]),
    "shaken_slab_exchange": (C.c_int, [_p]),
    "shaken_test_band_hook": (C.c_int, [_p, C.c_int, C.c_uint32]),
    "shaken_static_setup": (C.c_int, []),
    "shaken_run_static": (C.c_int, [_p, _p, C.c_int32, C.c_int32, C.c_uint64, C.c_uint64, C.c_double, C.c_double,
                                    C.c_int64, C.c_int64, _p, C.c_int64, _p]),
    "shaken_moments": (C.c_int, [_p, C.c_int64, C.c_int64, C.c_int64, C.POINTER(C.c_double)]),
    "shaken_selftest_philox_rate": (C.c_int, [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_double)]),
    "shaken_last_error": (C.c_char_p, [_p]),
    "shaken_version": (C.c_char_p, []),
}

_lib = None


class ShakenError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libshaken error {code}: {msg}")
        self.code = code


def lib():
    """Load libshaken.so (built by ``python -m paper_1908_07341_b200.build``).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1908_07341_b200.build` "
                "(nvcc, sm_100a).  libshaken has no CPU fallback."
            )
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def version() -> str:
    return lib().shaken_version().decode()


def alt_thresholds(J: float) -> np.ndarray:
    """Host-side integer acceptance table A[k] of the alternate dynamics (shaken_alt_thresholds)."""
    t = (C.c_uint32 * 5)()
    rc = lib().shaken_alt_thresholds(float(J), t)
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())
    return np.array(list(t), dtype=np.uint32)


def thresholds(J: float, q: float) -> np.ndarray:
    """Host-side integer acceptance table T[2k+c] (shaken_thresholds)."""
    t = (C.c_uint32 * 6)()
    rc = lib().shaken_thresholds(float(J), float(q), t)
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())
    return np.array(list(t), dtype=np.uint32)


def philox_only_rate(blocks_per_sm: int = 8, iters: int = 2048, reps: int = 3) -> float:
    """Measured rate (site-updates per ns) of the library's Philox-only kernel (shaken_selftest_philox_rate)."""
    v = C.c_double()
    rc = lib().shaken_selftest_philox_rate(int(blocks_per_sm), int(iters), int(reps), C.byref(v))
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())
    return float(v.value)


STATIC_SCRATCH_BYTES = 2621440     # SHAKEN_STATIC_SCRATCH_BYTES of include/shaken.h


def static_setup() -> None:
    """shaken_static_setup: once per device, with that device current (looks up the static scratch array's address)."""
    rc = lib().shaken_static_setup()
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())


def run_static(sigma_ptr: int, tau_ptr: int, L: int, n_chains: int, seed: int, t0: int, J: float, q: float,
               n_steps: int, obs_every: int = 0, rec_ptr: int = 0, max_records: int = 0, stream_ptr: int = 0) -> None:
    """shaken_run_static: n_steps of the shaken dynamics on caller-owned DEVICE buffers (int8 sigma, tau; int64 records),
    one cooperative launch, no allocation (the scratch is a static device array shared by all calls on the device)."""
    rc = lib().shaken_run_static(int(sigma_ptr), int(tau_ptr), int(L), int(n_chains), int(seed), int(t0), float(J), float(q),
                                 int(n_steps), int(obs_every), int(rec_ptr) or None, int(max_records), int(stream_ptr) or None)
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())


def philox_words(ctr: np.ndarray, key: np.ndarray) -> np.ndarray:
    """Device Philox4x32-10 of n (counter, key) pairs (test hook)."""
    c = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    k = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    assert c.shape[0] == k.shape[0]
    out = np.empty_like(c)
    rc = lib().shaken_philox_words(c.ctypes.data, k.ctypes.data, out.ctypes.data, c.shape[0])
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())
    return out


class Shaken:
    """One libshaken context: n_chains independent L x L tori."""

    def __init__(self, L: int, n_chains: int = 1, seed: int = 0, packed: bool = False,
                 use_torch: bool = True, max_records: int = 0, device: str = "cuda:0", stream=None):
        self.L, self.n_chains, self.seed, self.packed = int(L), int(n_chains), int(seed), bool(packed)
        self._h = _p()
        self._lib = lib()
        rc = self._lib.shaken_create(C.byref(self._h), self.L, self.n_chains, self.seed & (2**64 - 1),
                                     PACKED if packed else INT8)
        if rc:
            self._h = _p()
            raise ShakenError(rc, self._lib.shaken_last_error(None).decode())
        self._tensors = None
        if use_torch:
            import torch

            if not torch.cuda.is_available():
                self.close()
                raise RuntimeError("libshaken needs a CUDA device (there is no CPU fallback)")
            dev = torch.device(device)
            nb = int(self._lib.shaken_spin_bytes(self._h))
            with torch.cuda.device(dev):
                sigma = torch.empty(nb, dtype=torch.int8, device=dev)
                tau = torch.empty(nb, dtype=torch.int8, device=dev)
                rec = torch.zeros(max(int(max_records), 1) * self.n_chains * N_OBS, dtype=torch.int64, device=dev)
                st = stream if stream is not None else torch.cuda.current_stream(dev)
                self._tensors = (sigma, tau, rec, st)
                self._ck(self._lib.shaken_bind(self._h, sigma.data_ptr(), tau.data_ptr(), rec.data_ptr(),
                                               rec.numel() * 8, st.cuda_stream))
        elif max_records:
            self._ck(self._lib.shaken_reserve_records(self._h, int(max_records)))

    # ------------------------------------------------------------------ plumbing
    def _ck(self, rc):
        if rc < 0:
            raise ShakenError(int(rc), self._lib.shaken_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._lib.shaken_destroy(self._h)
            self._h = _p()
        self._tensors = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    @property
    def n_sites(self) -> int:
        return self.L * self.L

    @property
    def torch_tensors(self):
        """(sigma, tau, records, stream) borrowed by the library, or None."""
        return self._tensors

    # ------------------------------------------------------------------ the calls of include/shaken.h
    def init(self, mode: int):
        self._ck(self._lib.shaken_init(self._h, int(mode)))

    def run(self, J: float, q: float, n_steps: int, obs_every: int = 0):
        self._ck(self._lib.shaken_run(self._h, float(J), float(q), int(n_steps), int(obs_every)))

    def run_grid(self, J, q, n_steps: int, obs_every: int = 0):
        Ja = np.ascontiguousarray(J, dtype=np.float64)
        qa = np.ascontiguousarray(q, dtype=np.float64)
        if Ja.shape != (self.n_chains,) or qa.shape != (self.n_chains,):
            raise ValueError("J and q must have one entry per chain")
        self._ck(self._lib.shaken_run_grid(self._h, Ja.ctypes.data, qa.ctypes.data, int(n_steps), int(obs_every)))

    def run_alternate(self, J, n_steps: int, obs_every: int = 0):
        """Alternate (even sites, then odd sites) heat bath on sigma (shaken_run_alternate[_grid]); J scalar or per chain."""
        if np.ndim(J) == 0:
            self._ck(self._lib.shaken_run_alternate(self._h, float(J), int(n_steps), int(obs_every)))
            return
        Ja = np.ascontiguousarray(J, dtype=np.float64)
        if Ja.shape != (self.n_chains,):
            raise ValueError("J must have one entry per chain")
        self._ck(self._lib.shaken_run_alternate_grid(self._h, Ja.ctypes.data, int(n_steps), int(obs_every)))

    def observables(self, max_records: Optional[int] = None, out: Optional[np.ndarray] = None) -> np.ndarray:
        n = int(self._ck(self._lib.shaken_num_records(self._h)))
        if max_records is not None:
            n = min(n, int(max_records))
        if out is None:
            out = np.zeros((n, self.n_chains, N_OBS), dtype=np.int64)
        got = self._ck(self._lib.shaken_observables(self._h, out.ctypes.data, n))
        return out[:got]

    @property
    def num_records(self) -> int:
        return int(self._ck(self._lib.shaken_num_records(self._h)))

    def clear_records(self):
        self._ck(self._lib.shaken_clear_records(self._h))

    def get_spins(self, which: int, out: Optional[np.ndarray] = None) -> np.ndarray:
        if out is None:
            out = np.empty((self.n_chains, self.L, self.L), dtype=np.int8)
        assert out.dtype == np.int8 and out.size == self.n_chains * self.n_sites and out.flags.c_contiguous
        self._ck(self._lib.shaken_get_spins(self._h, int(which), out.ctypes.data))
        return out

    def set_spins(self, which: int, spins: np.ndarray):
        s = np.ascontiguousarray(spins, dtype=np.int8)
        if s.size != self.n_chains * self.n_sites:
            raise ValueError("wrong number of spins")
        self._ck(self._lib.shaken_set_spins(self._h, int(which), s.ctypes.data))

    def get_spins_into(self, which: int, host_ptr: int):
        """Raw-pointer form (e.g. a pinned torch tensor's data_ptr())."""
        self._ck(self._lib.shaken_get_spins(self._h, int(which), host_ptr))

    def set_spins_from(self, which: int, host_ptr: int):
        self._ck(self._lib.shaken_set_spins(self._h, int(which), host_ptr))

    def observables_into(self, host_ptr: int, max_records: int) -> int:
        return int(self._ck(self._lib.shaken_observables(self._h, host_ptr, int(max_records))))

    @property
    def step(self) -> int:
        v = C.c_uint64()
        self._ck(self._lib.shaken_get_step(self._h, C.byref(v)))
        return int(v.value)

    @step.setter
    def step(self, v: int):
        self._ck(self._lib.shaken_set_step(self._h, int(v)))

    def set_chain_offset(self, first_chain: int):
        self._ck(self._lib.shaken_set_chain_offset(self._h, int(first_chain)))

    def set_coupling(self, group: int):
        self._ck(self._lib.shaken_set_coupling(self._h, int(group)))
        self.group = int(group)

    def coalescence(self) -> np.ndarray:
        """Coalescence time of every coupling group in full steps, -1 = not yet (empty when uncoupled)."""
        g = getattr(self, "group", 1)
        ng = self.n_chains // g if g > 1 else 0
        out = np.full(ng, -1, dtype=np.int64)
        got = self._ck(self._lib.shaken_coalescence(self._h, out.ctypes.data, ng))
        return out[:got]

    def diag_correlations(self, ells) -> np.ndarray:
        """[chain][ell][2] int64: translation-summed SW-NE and NW-SE diagonal products of the current sigma."""
        e = np.ascontiguousarray(ells, dtype=np.int32)
        out = np.zeros((self.n_chains, e.size, 2), dtype=np.int64)
        self._ck(self._lib.shaken_diag_correlations(self._h, e.ctypes.data, e.size, out.ctypes.data))
        return out

    def test_band_hook(self, what: int, value: int):
        self._ck(self._lib.shaken_test_band_hook(self._h, int(what), int(value)))

    def adopt_spins(self):
        """Declare that the bound device buffers already hold valid spins (shaken_adopt_spins)."""
        self._ck(self._lib.shaken_adopt_spins(self._h))

    def synchronize(self):
        self._ck(self._lib.shaken_synchronize(self._h))

    @property
    def launch_count(self) -> int:
        return int(self._lib.shaken_launch_count(self._h))

    def set_variant(self, v: int):
        self._ck(self._lib.shaken_set_variant(self._h, int(v)))


class ShakenSlab(Shaken):
    """Rows [row0, row0 + n_rows) of one L x L lattice (shaken_create_slab): one slab of a row-slab sharded run.  The
    library owns the device buffers; spins move as [n_rows, L] arrays; records are the slab's partial sums."""

    def __init__(self, L: int, row0: int, n_rows: int, seed: int = 0, max_records: int = 0, stream=None):
        self.L, self.n_chains, self.seed, self.packed = int(L), 1, int(seed), False
        self.row0, self.n_rows = int(row0), int(n_rows)
        self._h = _p()
        self._lib = lib()
        self._tensors = None
        rc = self._lib.shaken_create_slab(C.byref(self._h), self.L, self.row0, self.n_rows, self.seed & (2**64 - 1))
        if rc:
            self._h = _p()
            raise ShakenError(rc, self._lib.shaken_last_error(None).decode())
        if stream is not None:
            self._ck(self._lib.shaken_set_stream(self._h, stream.cuda_stream))
            self._tensors = (None, None, None, stream)          # keeps the stream alive
        if max_records:
            self._ck(self._lib.shaken_reserve_records(self._h, int(max_records)))

    @property
    def n_sites(self) -> int:
        return self.n_rows * self.L

    def get_spins(self, which: int, out: Optional[np.ndarray] = None) -> np.ndarray:
        if out is None:
            out = np.empty((self.n_rows, self.L), dtype=np.int8)
        return super().get_spins(which, out)

    def inbox(self) -> int:
        ptr, nb = _p(), C.c_size_t()
        self._ck(self._lib.shaken_slab_inbox(self._h, C.byref(ptr), C.byref(nb)))
        return int(ptr.value)

    def connect(self, below_inbox: int, above_inbox: int):
        self._ck(self._lib.shaken_slab_connect(self._h, _p(below_inbox), _p(above_inbox)))

    def ipc_export(self) -> bytes:
        buf = C.create_string_buffer(64)
        self._ck(self._lib.shaken_slab_ipc_export(self._h, buf))
        return buf.raw

    def ipc_connect(self, below_handle: bytes, above_handle: bytes):
        self._ck(self._lib.shaken_slab_ipc_connect(self._h, C.c_char_p(below_handle), C.c_char_p(above_handle)))

    def exchange(self):
        self._ck(self._lib.shaken_slab_exchange(self._h))


# ---------------------------------------------------------------------- (a9) derived statistics, host side
def derived_stats(M, n_sites: int) -> dict:
    """Mean and variance of the magnetisation m = M / n_sites over the recorded window, plus <|m|>,
    <m^2>, <m^4> and the Binder cumulant U = 1 - <m^4> / (3 <m^2>^2): shaken_moments of the C ABI (exact integer power
    sums in the library -- M^4 overflows int64 from L = 512 on -- and one division each); this only marshals."""
    vals = np.ascontiguousarray(np.asarray(M).ravel(), dtype=np.int64)
    if vals.size == 0:
        raise ValueError("no records")
    out = (C.c_double * 6)()
    rc = lib().shaken_moments(vals.ctypes.data, vals.size, 1, int(n_sites), out)
    if rc:
        raise ShakenError(rc, lib().shaken_last_error(None).decode())
    return {"n": int(vals.size), "m": out[0], "abs_m": out[1], "m2": out[2], "m4": out[3], "var_m": out[4], "binder": out[5]}


def energy(J: float, q: float, E_J: int, E_q: int) -> float:
    """H(sigma, tau) = -(J E_J + q E_q), eq. (5)."""
    return -(float(J) * float(int(E_J)) + float(q) * float(int(E_q)))
