"""CPU-only checks of the boundary: the C-ABI library loads, exports every symbol include/shaken.h declares,
and its host-side logic (argument validation, threshold table, derived statistics) behaves as documented.
No compute call is made here (there is no GPU in this container)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1908_07341_b200 import shaken, workloads
from tests import pins

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "shaken.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(shaken_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = shaken.lib()
    names = declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    # and the binding knows every one of them (same names on both sides)
    assert set(names) == set(shaken.SIGNATURES)
    assert "sm_100a" in shaken.version()


def test_create_validates_arguments_without_a_device():
    lib = shaken.lib()
    h = C.c_void_p()
    for L, n, flags in [(15, 1, 0), (24, 1, 0), (48, 1, 1), (8, 1, 0), (65552, 1, 0), (64, 0, 0), (64, 1, 7)]:
        assert lib.shaken_create(C.byref(h), L, n, 1, flags) == shaken.EINVAL, (L, n, flags)
        assert not h.value
        assert lib.shaken_last_error(None) != b""
    assert lib.shaken_create(C.byref(h), 48, 3, 1, 0) == 0
    assert lib.shaken_spin_bytes(h) == 3 * 48 * 48
    assert lib.shaken_record_bytes(h) == 3 * 6 * 8
    assert lib.shaken_num_records(h) == 0
    step = C.c_uint64(99)
    assert lib.shaken_get_step(h, C.byref(step)) == 0 and step.value == 0
    assert lib.shaken_set_step(h, 12345678901234) == 0
    assert lib.shaken_get_step(h, C.byref(step)) == 0 and step.value == 12345678901234
    # run before any spins exist: ESTATE, not a crash; bad couplings: EINVAL
    assert lib.shaken_run(h, 0.5, float("nan"), 1, 0) == shaken.EINVAL
    assert lib.shaken_run(h, 0.5, 0.5, -1, 0) == shaken.EINVAL
    assert lib.shaken_run(h, 0.5, 0.5, 1, 0) == shaken.ESTATE
    assert b"no sigma" in lib.shaken_last_error(h)
    assert lib.shaken_adopt_spins(h) == shaken.ESTATE          # no buffers bound
    assert lib.shaken_set_variant(h, 5) == shaken.EINVAL and lib.shaken_set_variant(h, 3) == 0 and lib.shaken_set_variant(h, 0) == 0
    assert lib.shaken_run_alternate(h, float("inf"), 1, 0) == shaken.EINVAL
    assert lib.shaken_run_alternate(h, 0.3, 1, -2) == shaken.EINVAL
    assert lib.shaken_run_alternate(h, 0.3, 1, 0) == shaken.ESTATE
    assert lib.shaken_run_alternate_grid(h, None, 1, 0) == shaken.EINVAL
    assert lib.shaken_bind(h, None, None, None, 0, None) == shaken.EINVAL
    assert lib.shaken_destroy(h) == 0
    assert lib.shaken_create(C.byref(h), 64, 2, 1, 1) == 0
    assert lib.shaken_spin_bytes(h) == 2 * 64 * 64 // 8
    assert lib.shaken_destroy(h) == 0


COUPLINGS = [(0.5, 0.5), (0.6585, 0.6585), (0.7, 0.7), (0.45, 10.0), (0.44, 0.66), (1.2, 20.0), (0.0, 0.0),
             (0.0, 1.0), (1.0, 0.0), (-0.3, 0.4), (2.0, 0.03)]


def test_slab_and_hook_arguments_are_validated_without_a_device():
    lib = shaken.lib()
    h = C.c_void_p()
    for L, row0, n in [(24, 0, 8), (64, -1, 8), (64, 0, 1), (64, 60, 8), (65552, 0, 8)]:
        assert lib.shaken_create_slab(C.byref(h), L, row0, n, 1) == shaken.EINVAL, (L, row0, n)
        assert not h.value
    assert lib.shaken_create_slab(C.byref(h), 64, 16, 32, 1) == 0
    assert lib.shaken_spin_bytes(h) == 32 * 64                      # the slab's own rows
    assert lib.shaken_record_bytes(h) == 6 * 8
    assert lib.shaken_bind(h, C.c_void_p(16), C.c_void_p(32), None, 0, None) == shaken.ESTATE   # a slab owns its buffers
    assert lib.shaken_run(h, 0.5, 0.5, 1, 0) == shaken.ESTATE       # no sigma yet
    assert lib.shaken_run_alternate(h, 0.5, 1, 0) == shaken.ESTATE
    assert lib.shaken_slab_connect(h, None, None) == shaken.EINVAL
    assert lib.shaken_test_band_hook(h, 7, 0) == shaken.EINVAL
    assert lib.shaken_destroy(h) == 0
    assert lib.shaken_create(C.byref(h), 64, 1, 1, 0) == 0
    assert lib.shaken_slab_exchange(h) == shaken.EINVAL             # not a slab context
    assert lib.shaken_slab_connect(h, C.c_void_p(16), C.c_void_p(16)) == shaken.EINVAL
    assert lib.shaken_destroy(h) == 0


def test_library_threshold_table_against_exact_decimal_arithmetic():
    """The library's own host table (not the oracle's) against 60-digit decimal evaluation of
    round(2^32 e^h / (2 cosh h)) -- same pin as the oracle's, applied independently."""
    for J, q in COUPLINGS:
        T = shaken.thresholds(J, q)
        ex = pins.exact_table(J, q)
        for i in range(6):
            if int(T[i]) != int(ex[i]):
                frac = float(pins.exact_threshold_real(pins.field(J, q, i // 2, i % 2)) % 1)
                assert abs(frac - 0.5) < 4e-6 and abs(int(T[i]) - int(ex[i])) == 1
        assert int(T[0]) + int(T[5]) == 2**32 and int(T[1]) + int(T[4]) == 2**32 and int(T[2]) + int(T[3]) == 2**32
    J, q = workloads.grid_couplings()
    for a, b in list(zip(J, q))[::37]:
        assert np.array_equal(shaken.thresholds(a, b).astype(np.uint64), pins.exact_table(a, b))
    with pytest.raises(shaken.ShakenError):
        shaken.thresholds(float("inf"), 0.1)


def test_moments_through_the_c_abi_strided_and_beyond_128_bits():
    """shaken_moments as a C caller uses it: a strided view into [record][chain][6] records, and a window whose sum of
    M^4 exceeds 128 bits (500 records of |M| = 2^32 - 2k on a 65536^2 lattice); expected values from Python integers
    and Fractions written out here (not from either implementation's code)."""
    from fractions import Fraction

    lib = shaken.lib()
    rec = np.zeros((5, 3, 6), dtype=np.int64)
    rec[:, 1, 0] = [2, -2, 4, 0, 4]
    out = (C.c_double * 6)()
    assert lib.shaken_moments(rec[0, 1].ctypes.data, 4, 18, 4, out) == 0          # first four records of chain 1
    assert list(out) == [0.25, 0.5, 0.375, 0.28125, 0.3125, out[5]] and abs(out[5] - 1 / 3) < 1e-15
    N = 2**32
    M = np.array([(N - 2 * k) * (1 if k % 3 else -1) for k in range(500)], dtype=np.int64)
    assert lib.shaken_moments(M.ctypes.data, 500, 1, N, out) == 0
    Mi = [int(v) for v in M]
    S1, Sa, S2, S4 = sum(Mi), sum(abs(v) for v in Mi), sum(v * v for v in Mi), sum(v**4 for v in Mi)
    assert S4 > 2**128
    want = [Fraction(S1, 500 * N), Fraction(Sa, 500 * N), Fraction(S2, 500 * N * N), Fraction(S4, 500 * N**4),
            Fraction(500 * S2 - S1 * S1, 500 * 500 * N * N), 1 - Fraction(500 * S4, 3 * S2 * S2)]
    for got, w in zip(out, want):
        assert abs(got - float(w)) <= 1e-15 * abs(float(w)), (got, float(w))
    # U < 0 (one large outlier among zeros): the sign branch of the 256-bit subtraction
    assert lib.shaken_moments(np.array([8, 0, 0, 0, 0, 0, 0, 0], dtype=np.int64).ctypes.data, 8, 1, 64, out) == 0
    assert abs(out[5] - (1 - 8 / 3)) < 1e-15
    assert np.isnan(shaken.derived_stats([0, 0], 16)["binder"])
    for bad in [(0, 1, 4), (4, 0, 4), (4, 1, 0), (4, 1, 3)]:                       # n, stride, n_sites (|M| = 4 > 3)
        assert lib.shaken_moments(rec[0, 1].ctypes.data, bad[0], bad[1] * 18, bad[2], out) == shaken.EINVAL, bad
    assert lib.shaken_moments(None, 4, 1, 4, out) == shaken.EINVAL


def test_derived_stats_exact_small_case_and_large_values():
    """(a9) host statistics: hand-computed case, and no overflow where M^4 exceeds int64 (L >= 512)."""
    st = shaken.derived_stats([2, -2, 4, 0], 4)
    assert st["m"] == 0.25 and st["abs_m"] == 0.5 and st["m2"] == 24 / (4 * 16) and st["m4"] == (16 + 16 + 256) / (4 * 256)
    assert st["var_m"] == 24 / 64 - 0.25**2
    assert abs(st["binder"] - (1 - st["m4"] / (3 * st["m2"] ** 2))) < 1e-15
    N = 32768 * 32768
    M = [N, N - 2, -(N - 4)]
    st = shaken.derived_stats(M, N)
    assert abs(st["m4"] - 1.0) < 1e-8 and abs(st["abs_m"] - 1.0) < 1e-8
    assert abs(st["binder"] - 2.0 / 3.0) < 1e-8
    assert shaken.energy(0.5, 2.0, 10, -3) == -(0.5 * 10 + 2.0 * -3)


def test_header_compiles_as_c99_and_a_c_caller_links(tmp_path):
    """include/shaken.h is a C header (no C++ types): a C99 program that includes it compiles with -pedantic, links against
    libshaken.so and gets the host-side results (thresholds, moments) without a device."""
    import shutil
    import subprocess

    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("gcc not found")
    src = tmp_path / "caller.c"
    src.write_text("""
#include "shaken.h"
#include <stdio.h>
int main(void) {
    uint32_t t[6]; double m[SHAKEN_N_MOMENTS]; int64_t M[3] = {4, -4, 0};
    if (shaken_thresholds(0.0, 0.0, t) != SHAKEN_OK) return 1;
    if (shaken_moments(M, 3, 1, 16, m) != SHAKEN_OK) return 2;
    printf("%u %.6f %.6f\\n", t[0], m[2], m[5]);
    return 0;
}
""")
    exe = tmp_path / "caller"
    libdir = os.path.dirname(shaken.LIB_PATH)
    subprocess.check_call([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe),
                           "-L", libdir, "-l:libshaken.so", f"-Wl,-rpath,{libdir}"])
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    assert out[0] == str(2**31)                     # T(0) = 2^31
    assert abs(float(out[1]) - (32 / 3) / 256) < 1e-6 and abs(float(out[2]) - 0.5) < 1e-6
