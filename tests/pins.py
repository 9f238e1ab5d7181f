"""Independent pins used by the ``-m "not gpu"`` tests: none of this calls the oracle or the CUDA path.

* :func:`curand_host_words`  -- Philox4x32-10 words produced by cuRAND's HOST generator (a library routine;
  runs on the CPU, no GPU needed).  Layout found by probing the library: output group ``g`` (4 words) of a
  generator with seed ``S`` and offset ``4*65536*k`` is Philox(counter=(k lo32, k hi32, g % 65536, 0), key=S)
  for ``g < 65536``.
* :func:`exact_threshold`    -- round(2^32 / (1 + exp(-2h))) in 60-digit decimal arithmetic (closed form of
  P(+|h) = e^h / (2 cosh h)).
* :func:`brute_half_step`    -- eq. (15)/(16) of PAPER.md:162-172 on a tiny torus with numpy ``roll``.
* :func:`brute_observables`  -- the six sums with numpy ``roll`` (eq. 5 :81-84, eq. 17 :196).
* :func:`exact_kernels_3x3`  -- the 512x512 transition matrices of eq. (15) and (16) on the 3x3 torus.
"""
from __future__ import annotations

import ctypes as C
import glob
import os
from decimal import Decimal, getcontext

import numpy as np

getcontext().prec = 60


# ----------------------------------------------------------------------------- cuRAND host generator
def _find_curand():
    cands = ["/usr/local/cuda/lib64/libcurand.so.10", "/usr/local/cuda/lib64/libcurand.so"]
    try:
        import nvidia.curand  # type: ignore

        for base in nvidia.curand.__path__:
            cands += glob.glob(os.path.join(base, "lib", "libcurand.so*"))
    except Exception:
        pass
    for p in cands:
        if os.path.exists(p):
            try:
                return C.CDLL(p)
            except OSError:
                continue
    return None


_curand = None


def curand_available() -> bool:
    global _curand
    if _curand is None:
        _curand = _find_curand() or False
    return bool(_curand)


def curand_host_stream(seed: int, k: int, n_groups: int) -> np.ndarray:
    """Groups g = 0..n_groups-1 (n_groups <= 65536) for counter (k lo, k hi, g, 0); shape [n_groups, 4]."""
    assert curand_available() and 0 < n_groups <= 65536
    cur = _curand
    gen = C.c_void_p()
    assert cur.curandCreateGeneratorHost(C.byref(gen), 161) == 0  # CURAND_RNG_PSEUDO_PHILOX4_32_10
    try:
        assert cur.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed & (2**64 - 1))) == 0
        assert cur.curandSetGeneratorOffset(gen, C.c_ulonglong((4 * 65536 * k) & (2**64 - 1))) == 0
        out = np.zeros(4 * n_groups, dtype=np.uint32)
        assert cur.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(out.size)) == 0
    finally:
        cur.curandDestroyGenerator(gen)
    return out.reshape(n_groups, 4)


def curand_site_words(seed: int, chain: int, g: int, n_sites: int) -> np.ndarray:
    """Random word of every site for half-step index g (< 65536) of one chain, taken from cuRAND:
    counter = (site>>2, chain, g, 0), word site&3  (the mapping DESIGN.md fixes)."""
    assert 0 <= g < 65536
    words = np.zeros(n_sites, dtype=np.uint32)
    n_calls = (n_sites + 3) // 4
    for call in range(n_calls):
        k = call + (chain << 32)
        grp = curand_host_stream(seed, k, g + 1)[g]
        lo = 4 * call
        hi = min(n_sites, lo + 4)
        words[lo:hi] = grp[: hi - lo]
    return words


# ----------------------------------------------------------------------------- thresholds, exact
def exact_p_plus(h: float) -> Decimal:
    """P(+|h) = e^h/(2 cosh h) = 1/(1+e^{-2h}) with the double h taken exactly."""
    return Decimal(1) / (Decimal(1) + (Decimal(-2) * Decimal(h)).exp())


def exact_threshold_real(h: float) -> Decimal:
    return exact_p_plus(h) * Decimal(2**32)


def exact_threshold(h: float) -> int:
    """Nearest integer to 2^32 P(+|h), mirrored for h<0, clamped to [1, 2^32-1] (reading 7)."""
    def F(a):
        v = int((exact_threshold_real(a) + Decimal("0.5")).to_integral_value(rounding="ROUND_FLOOR"))
        return min(max(v, 2**31), 2**32 - 1)

    return F(h) if h >= 0 else 2**32 - F(-h)


def field(J: float, q: float, k: int, c: int) -> float:
    """eq. (14): h = J*(sum of the two J-neighbours) + q*self, with k = #(+1 neighbours), c = [self=+1]."""
    return float(2 * k - 2) * J + float(2 * c - 1) * q


def exact_table(J: float, q: float) -> np.ndarray:
    return np.array([exact_threshold(field(J, q, k, c)) for k in range(3) for c in range(2)], dtype=np.uint64)


# ----------------------------------------------------------------------------- brute force on small tori
def brute_half_step(src: np.ndarray, half: int, table, words: np.ndarray) -> np.ndarray:
    """src: [L, L] int8 indexed [r, c].  half 0: neighbours down (r-1) and left (c-1)  (eq. 15, Alg. 2);
    half 1: up (r+1) and right (c+1) (eq. 16, Alg. 1).  words: [L*L] uint32 in site order r*L+c."""
    L = src.shape[0]
    if half == 0:
        vert = np.roll(src, 1, axis=0)   # vert[r] = src[r-1]
        horz = np.roll(src, 1, axis=1)   # horz[:, c] = src[:, c-1]
    else:
        vert = np.roll(src, -1, axis=0)  # src[r+1]
        horz = np.roll(src, -1, axis=1)  # src[:, c+1]
    k = (vert == 1).astype(np.int64) + (horz == 1).astype(np.int64)
    idx = 2 * k + (src == 1)
    T = np.asarray(table, dtype=np.uint64)[idx]
    w = words.reshape(L, L).astype(np.uint64)
    return np.where(w < T, 1, -1).astype(np.int8)


def brute_observables(sigma: np.ndarray, tau: np.ndarray) -> np.ndarray:
    s = sigma.astype(np.int64)
    t = tau.astype(np.int64)
    t_up, t_right = np.roll(t, -1, axis=0), np.roll(t, -1, axis=1)
    s_up, s_right = np.roll(s, -1, axis=0), np.roll(s, -1, axis=1)
    return np.array(
        [s.sum(), t.sum(), (s * (t_up + t_right)).sum(), (s * t).sum(), (s * s_right).sum(), (s * s_up).sum()],
        dtype=np.int64,
    )


# ----------------------------------------------------------------------------- exact 3x3 kernels
def all_configs(L: int = 3) -> np.ndarray:
    """[2^(L*L), L, L] int8; configuration number n has spin +1 at site x iff bit x of n is set."""
    n = L * L
    ids = np.arange(2**n, dtype=np.int64)
    bits = (ids[:, None] >> np.arange(n)[None, :]) & 1
    return (2 * bits - 1).astype(np.int8).reshape(-1, L, L)


def config_id(cfg: np.ndarray) -> np.ndarray:
    """Inverse of all_configs for an array [..., L, L]."""
    L = cfg.shape[-1]
    b = (cfg.reshape(*cfg.shape[:-2], L * L) == 1).astype(np.int64)
    return (b << np.arange(L * L)).sum(axis=-1)


def exact_kernels_3x3(J: float, q: float, table=None):
    """P15[s, t] = P(tau'=t | sigma=s) of eq. (15), P16[t, s'] = P(sigma'=s' | tau=t) of eq. (16) on the 3x3 torus.
    With ``table`` (six integer thresholds) the per-site probability is T/2^32 instead of e^h/(2 cosh h).
    Also returns Z_sigma = prod_x 2 cosh(h_left_down_x(sigma))."""
    cfgs = all_configs(3).astype(np.float64)
    n = cfgs.shape[0]

    def fields(c, half):
        if half == 0:
            return J * (np.roll(c, 1, axis=1) + np.roll(c, 1, axis=2)) + q * c    # down + left
        return J * (np.roll(c, -1, axis=1) + np.roll(c, -1, axis=2)) + q * c      # up + right

    def p_plus(c, half):
        h = fields(c, half)
        if table is None:
            return np.exp(h) / (2.0 * np.cosh(h))
        if half == 0:
            k = (np.roll(c, 1, axis=1) == 1).astype(int) + (np.roll(c, 1, axis=2) == 1).astype(int)
        else:
            k = (np.roll(c, -1, axis=1) == 1).astype(int) + (np.roll(c, -1, axis=2) == 1).astype(int)
        idx = 2 * k + (c == 1)
        return np.asarray(table, dtype=np.float64)[idx] / 2.0**32

    out = []
    for half in (0, 1):
        pp = p_plus(cfgs, half).reshape(n, 1, 9)            # source config, site
        tgt = (cfgs.reshape(1, n, 9) == 1)                  # target config, site
        probs = np.where(tgt, pp, 1.0 - pp)                 # [src, tgt, site]
        out.append(probs.prod(axis=2))
    Zs = (2.0 * np.cosh(fields(cfgs, 0))).reshape(n, 9).prod(axis=1)
    return out[0], out[1], Zs


def hamiltonian_pair(sigma: np.ndarray, tau: np.ndarray, J: float, q: float) -> float:
    """H(sigma, tau), first form of eq. (5)."""
    s = sigma.astype(np.float64)
    t = tau.astype(np.float64)
    return float(-(J * s * (np.roll(t, -1, axis=0) + np.roll(t, -1, axis=1)) + q * s * t).sum())
