"""ctypes wrapper around oracle/shaken_oracle.c -- ORACLE (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` leg
may import this module.  It shares nothing with ``paper_1908_07341_b200`` and never imports it.

The arithmetic lives in the C file (which cites PAPER.md passage by passage); this module only
marshals arguments and, in :func:`derived_stats`, turns int64 records into the double-precision
quantities of PAPER.md:194 (mean and variance of the magnetisation m, eq. 17 :196) plus
<|m|>, <m^2>, <m^4> and the Binder cumulant named by BASELINE.json, using exact Python integers and
ONE final division each (pinned by hand-computed records in tests/test_oracle_stats.py).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from fractions import Fraction

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "shaken_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

OBS_NAMES = ("M_sigma", "M_tau", "E_J", "E_q", "C_x", "C_y")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, no fast-math, no FP contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        p = C.c_void_p
        L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.oracle_philox4x32_10.restype = None
        L.oracle_threshold.argtypes = [C.c_double]
        L.oracle_threshold.restype = C.c_uint32
        L.oracle_thresholds.argtypes = [C.c_double, C.c_double, C.POINTER(C.c_uint32)]
        L.oracle_thresholds.restype = None
        L.oracle_create.argtypes = [C.POINTER(p), C.c_int64, C.c_int64, C.c_uint64]
        L.oracle_create.restype = C.c_int
        L.oracle_destroy.argtypes = [p]
        L.oracle_destroy.restype = None
        L.oracle_init.argtypes = [p, C.c_int]
        L.oracle_init.restype = C.c_int
        L.oracle_set_complement.argtypes = [p, C.c_int]
        L.oracle_set_complement.restype = None
        L.oracle_measure.argtypes = [p, p, C.c_int64, C.POINTER(C.c_int64)]
        L.oracle_measure.restype = None
        L.oracle_run.argtypes = [p, C.c_double, C.c_double, C.c_int64, C.c_int64]
        L.oracle_run.restype = C.c_int
        L.oracle_run_grid.argtypes = [p, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_int64, C.c_int64]
        L.oracle_run_grid.restype = C.c_int
        L.oracle_observables.argtypes = [p, C.POINTER(C.c_int64), C.c_int64]
        L.oracle_observables.restype = C.c_int64
        L.oracle_num_records.argtypes = [p]
        L.oracle_num_records.restype = C.c_int64
        L.oracle_get_spins.argtypes = [p, C.c_int, p]
        L.oracle_get_spins.restype = C.c_int
        L.oracle_set_spins.argtypes = [p, C.c_int, p]
        L.oracle_set_spins.restype = C.c_int
        L.oracle_get_step.argtypes = [p]
        L.oracle_get_step.restype = C.c_uint64
        L.oracle_set_step.argtypes = [p, C.c_uint64]
        L.oracle_set_step.restype = C.c_int
        L.oracle_half_step_rows.argtypes = [p, p, C.c_int64, C.c_uint64, C.c_int64, C.c_double, C.c_double,
                                            C.c_uint64, C.c_int, C.c_int64, C.c_int64]
        L.oracle_half_step_rows.restype = C.c_int
        L.oracle_diag_correlations.argtypes = [p, C.POINTER(C.c_int64), C.c_int64, C.POINTER(C.c_int64)]
        L.oracle_diag_correlations.restype = C.c_int
        L.oracle_alt_thresholds.argtypes = [C.c_double, C.POINTER(C.c_uint32)]
        L.oracle_alt_thresholds.restype = None
        L.oracle_alt_half_step_rows.argtypes = [p, p, C.c_int64, C.c_uint64, C.c_int64, C.c_double, C.c_uint64, C.c_int,
                                                C.c_int64, C.c_int64]
        L.oracle_alt_half_step_rows.restype = C.c_int
        L.oracle_run_alternate.argtypes = [p, C.POINTER(C.c_double), C.c_int64, C.c_int64]
        L.oracle_run_alternate.restype = C.c_int
        L.oracle_set_coupling.argtypes = [p, C.c_int64]
        L.oracle_set_coupling.restype = C.c_int
        L.oracle_coalescence.argtypes = [p, C.POINTER(C.c_int64), C.c_int64]
        L.oracle_coalescence.restype = C.c_int64
        _lib = L
    return _lib


def philox4x32_10(ctr, key):
    """Philox4x32-10 of one (counter, key); returns 4 uint32 as a numpy array."""
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def threshold(h: float) -> int:
    return int(lib().oracle_threshold(float(h)))


def thresholds(J: float, q: float) -> np.ndarray:
    t = (C.c_uint32 * 6)()
    lib().oracle_thresholds(float(J), float(q), t)
    return np.array(list(t), dtype=np.uint32)


def measure(sigma: np.ndarray, tau: np.ndarray) -> np.ndarray:
    """The six int64 sums of one (sigma, tau) pair of L x L int8 arrays."""
    s = np.ascontiguousarray(sigma, dtype=np.int8)
    t = np.ascontiguousarray(tau, dtype=np.int8)
    L = s.shape[-1]
    assert s.shape == (L, L) and t.shape == (L, L)
    out = (C.c_int64 * 6)()
    lib().oracle_measure(s.ctypes.data, t.ctypes.data, L, out)
    return np.array(list(out), dtype=np.int64)


def half_step_rows(src: np.ndarray, seed: int, chain: int, J: float, q: float, t: int, half: int,
                   r0: int, nrows: int) -> np.ndarray:
    """Rows r0 .. r0+nrows-1 of one half-step (0: eq. 15, 1: eq. 16) at full-step index t, computed from the
    full L x L source sublattice ``src`` (+-1 int8).  For spot checks at sizes where a whole step is too slow."""
    s = np.ascontiguousarray(src, dtype=np.int8)
    L = s.shape[-1]
    assert s.shape == (L, L)
    out = np.empty((nrows, L), dtype=np.int8)
    rc = lib().oracle_half_step_rows(s.ctypes.data, out.ctypes.data, L, int(seed) & 0xFFFFFFFFFFFFFFFF, int(chain),
                                     float(J), float(q), int(t), int(half), int(r0), int(nrows))
    if rc:
        raise OracleError(f"oracle_half_step_rows failed: {rc}")
    return out


def alt_thresholds(J: float) -> np.ndarray:
    """A[k], k = number of +1 among the four neighbours: alternate heat bath on the square lattice."""
    t = (C.c_uint32 * 5)()
    lib().oracle_alt_thresholds(float(J), t)
    return np.array(list(t), dtype=np.uint32)


def alt_half_step_rows(src: np.ndarray, seed: int, chain: int, J: float, t: int, half: int, r0: int,
                       nrows: int) -> np.ndarray:
    """Rows r0 .. r0+nrows-1 of the lattice after half-step ``half`` (0: even sites, 1: odd sites) of full step t of
    the alternate dynamics, from the full L x L lattice ``src`` before it."""
    s = np.ascontiguousarray(src, dtype=np.int8)
    L = s.shape[-1]
    assert s.shape == (L, L)
    out = np.empty((nrows, L), dtype=np.int8)
    rc = lib().oracle_alt_half_step_rows(s.ctypes.data, out.ctypes.data, L, int(seed) & 0xFFFFFFFFFFFFFFFF, int(chain),
                                         float(J), int(t), int(half), int(r0), int(nrows))
    if rc:
        raise OracleError(f"oracle_alt_half_step_rows failed: {rc}")
    return out


class OracleError(RuntimeError):
    pass


class Oracle:
    """Same calls as the library's context (create / init / run / observables / state I/O) on host memory."""

    def __init__(self, L: int, n_chains: int = 1, seed: int = 0):
        self.L, self.n_chains, self.seed = int(L), int(n_chains), int(seed)
        self._h = C.c_void_p()
        rc = lib().oracle_create(C.byref(self._h), self.L, self.n_chains, self.seed & 0xFFFFFFFFFFFFFFFF)
        if rc:
            raise OracleError(f"oracle_create failed: {rc}")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc, what):
        if rc:
            raise OracleError(f"{what} failed: {rc}")

    def init(self, mode: int):
        self._ck(lib().oracle_init(self._h, int(mode)), "oracle_init")

    def diag_correlations(self, ells) -> np.ndarray:
        """[chain][ell][2] int64: translation-summed SW-NE and NW-SE diagonal products of sigma."""
        e = np.ascontiguousarray(ells, dtype=np.int64)
        out = np.zeros((self.n_chains, e.size, 2), dtype=np.int64)
        self._ck(lib().oracle_diag_correlations(self._h, e.ctypes.data_as(C.POINTER(C.c_int64)), e.size,
                                                out.ctypes.data_as(C.POINTER(C.c_int64))), "oracle_diag_correlations")
        return out

    def set_coupling(self, group: int):
        """Chains c with equal c // group share their random numbers; forgets coalescence times."""
        self._ck(lib().oracle_set_coupling(self._h, int(group)), "oracle_set_coupling")
        self.group = int(group)

    def coalescence(self) -> np.ndarray:
        """Coalescence time of every group in full steps, -1 = not yet."""
        ng = self.n_chains // getattr(self, "group", 1) if getattr(self, "group", 1) > 1 else 0
        out = np.full(ng, -1, dtype=np.int64)
        if ng:
            got = lib().oracle_coalescence(self._h, out.ctypes.data_as(C.POINTER(C.c_int64)), ng)
            assert got == ng
        return out

    def set_complement(self, on: bool):
        lib().oracle_set_complement(self._h, int(bool(on)))

    def run(self, J: float, q: float, n_steps: int, obs_every: int = 0):
        self._ck(lib().oracle_run(self._h, float(J), float(q), int(n_steps), int(obs_every)), "oracle_run")

    def run_grid(self, J, q, n_steps: int, obs_every: int = 0):
        Ja = np.ascontiguousarray(J, dtype=np.float64)
        qa = np.ascontiguousarray(q, dtype=np.float64)
        assert Ja.shape == (self.n_chains,) and qa.shape == (self.n_chains,)
        self._ck(
            lib().oracle_run_grid(
                self._h,
                Ja.ctypes.data_as(C.POINTER(C.c_double)),
                qa.ctypes.data_as(C.POINTER(C.c_double)),
                int(n_steps),
                int(obs_every),
            ),
            "oracle_run_grid",
        )

    def run_alternate(self, J, n_steps: int, obs_every: int = 0):
        """Alternate (even sites, then odd sites) heat bath on the sigma array, coupling J (scalar or per chain)."""
        Ja = np.ascontiguousarray(np.broadcast_to(np.asarray(J, dtype=np.float64), (self.n_chains,)))
        self._ck(lib().oracle_run_alternate(self._h, Ja.ctypes.data_as(C.POINTER(C.c_double)), int(n_steps),
                                            int(obs_every)), "oracle_run_alternate")

    def observables(self) -> np.ndarray:
        n = int(lib().oracle_num_records(self._h))
        out = np.zeros((n, self.n_chains, 6), dtype=np.int64)
        if n:
            got = lib().oracle_observables(self._h, out.ctypes.data_as(C.POINTER(C.c_int64)), n)
            assert got == n
        return out

    def get_spins(self, which: int) -> np.ndarray:
        out = np.empty((self.n_chains, self.L, self.L), dtype=np.int8)
        self._ck(lib().oracle_get_spins(self._h, int(which), out.ctypes.data), "oracle_get_spins")
        return out

    def set_spins(self, which: int, spins: np.ndarray):
        s = np.ascontiguousarray(spins, dtype=np.int8).reshape(self.n_chains, self.L, self.L)
        self._ck(lib().oracle_set_spins(self._h, int(which), s.ctypes.data), "oracle_set_spins")

    @property
    def step(self) -> int:
        return int(lib().oracle_get_step(self._h))

    @step.setter
    def step(self, v: int):
        self._ck(lib().oracle_set_step(self._h, int(v)), "oracle_set_step")


def derived_stats(M, n_sites: int) -> dict:
    """<m>, <|m|>, <m^2>, <m^4>, Var m and Binder U = 1 - <m^4>/(3<m^2>^2) from the int64 magnetisation
    sums M (one per recorded step) of one chain.  Exact integer power sums, one division."""
    Ms = [int(v) for v in np.asarray(M).reshape(-1)]
    n = len(Ms)
    if n == 0:
        raise ValueError("no records")
    N = int(n_sites)
    S1 = sum(Ms)
    Sa = sum(abs(v) for v in Ms)
    S2 = sum(v * v for v in Ms)
    S4 = sum(v ** 4 for v in Ms)
    out = {
        "n": n,
        "m": float(Fraction(S1, n * N)),
        "abs_m": float(Fraction(Sa, n * N)),
        "m2": float(Fraction(S2, n * N * N)),
        "m4": float(Fraction(S4, n * N ** 4)),
        "var_m": float(Fraction(n * S2 - S1 * S1, n * n * N * N)),
    }
    out["binder"] = float(1 - Fraction(S4 * n, 3 * S2 * S2)) if S2 else float("nan")
    return out


def energy(J: float, q: float, E_J: int, E_q: int) -> float:
    """H(sigma, tau) of eq. (5): -(J*E_J + q*E_q)."""
    return -(float(J) * float(int(E_J)) + float(q) * float(int(E_q)))


# ---------------------------------------------------------------------- exact sampling
def propp_wilson(o: "Oracle", J, q=None, base: int = 1 << 40, max_doublings: int = 40):
    """Coupling from the past (Propp & Wilson 1996, the paper's ref. [13]; "two copies of the Markov
    chain ... run with the same update function and the same sequence of random numbers", :276 "samples are drawn
    using the Propp-Wilson algorithm"), written out step by step for a context whose coupling groups are pairs.

    Time runs over the NEGATIVE integers: the update from time s to s+1 always uses the random numbers of the full-step
    index ``base + s`` (counter-based generator: a fixed function of the index), whatever the starting time.  For
    T = 1, 2, 4, ...: start sigma^top (all +1) and sigma^bot (all -1) at time -T, run T steps to time 0; because the
    dynamics preserves the ordering (:238), once top and bottom agree at time 0 every start would have ended there and
    that configuration is an exact draw from the stationary measure.  All pairs are run with the same T until the last
    one has coalesced (a pair that coalesced from -T ends in the same state from any earlier start).

    q = None: the alternate heat bath on the square lattice (run_alternate) in place of the shaken dynamics; :276 draws
    the samples of that reference dynamics the same way.

    Returns (samples [n_pairs, L, L] int8 = sigma at time 0, T used)."""
    if getattr(o, "group", 1) != 2:
        raise ValueError("propp_wilson needs coupling groups of two (top, bottom)")
    Ja = np.ascontiguousarray(J, dtype=np.float64)
    qa = None if q is None else np.ascontiguousarray(q, dtype=np.float64)
    T = 1
    for _ in range(max_doublings):
        o.init(2)                       # top all +1, bottom all -1; also resets the step counter ...
        o.step = base - T               # ... so the starting time -T is set afterwards
        if qa is None:
            o.run_alternate(Ja, T, 0)
        else:
            o.run_grid(Ja, qa, T, 0)
        if np.all(o.coalescence() >= 0):
            return o.get_spins(0)[0::2].copy(), T
        T *= 2
    raise RuntimeError("no coalescence within the allowed number of doublings")
