"""pytest configuration: registers the ``gpu`` marker, puts the repo root on sys.path, makes sure the oracle's C
file is compiled (building the checker is not using it) and, when nvcc is present, that libshaken.so and the
test-only cuRAND reference are built in-tree (so they travel to the GPU box with the snapshot)."""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

HERE = os.path.dirname(os.path.abspath(__file__))
CURAND_REF_SRC = os.path.join(HERE, "curand_ref.cu")
CURAND_REF_LIB = os.path.join(HERE, "libcurandref.so")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running oracle comparison, excluded from the default CPU run")


def _nvcc():
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return None


def build_curand_ref():
    if os.path.exists(CURAND_REF_LIB) and os.path.getmtime(CURAND_REF_LIB) >= os.path.getmtime(CURAND_REF_SRC):
        return CURAND_REF_LIB
    nvcc = _nvcc()
    if nvcc is None:
        return None
    tmp = CURAND_REF_LIB + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, "-O2", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-shared",
                           "-cudart", "static", "-o", tmp, CURAND_REF_SRC])
    os.replace(tmp, CURAND_REF_LIB)
    return CURAND_REF_LIB


@pytest.fixture(scope="session", autouse=True)
def _build_native():
    from oracle import shaken_oracle

    shaken_oracle.build()
    if _nvcc() is not None:
        from paper_1908_07341_b200 import build as b

        b.build()
        build_curand_ref()
    yield


def has_gpu() -> bool:
    try:
        import torch

        return torch.cuda.is_available()
    except Exception:
        return False
