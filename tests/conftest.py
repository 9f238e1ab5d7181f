"""pytest configuration: registers the ``gpu`` marker, puts the repo root on sys.path and makes sure
the oracle's C file is compiled (building the checker is not using it)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running oracle comparison, excluded from the default CPU run")


@pytest.fixture(scope="session", autouse=True)
def _build_oracle():
    from oracle import shaken_oracle

    shaken_oracle.build()
    yield
