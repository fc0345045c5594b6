import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running CPU test")


@pytest.fixture(scope="session", autouse=True)
def _native_pieces_built():
    """Build the CUDA engine (nvcc, sm_100a) and the C oracle (gcc) once per session if they are
    missing or older than their sources; the binding itself never builds and never falls back."""
    from paper_2606_10440_b200 import build as engine_build
    from oracle import oracle
    engine_build.build()
    oracle.build()
