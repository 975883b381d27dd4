"""Shared fixtures.  `-m "not gpu"` runs here on CPU; `-m gpu` runs on a B200 through the C ABI."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def synth():
    from paper_2606_27262_b200 import synth as s
    s.build()
    return s


@pytest.fixture(scope="session")
def api():
    """The ctypes binding over libspt.so, built in-tree with nvcc (cross-compiles without a GPU)."""
    from paper_2606_27262_b200 import build
    build.build()
    from paper_2606_27262_b200 import api as a
    a.lib()
    return a


@pytest.fixture(scope="session")
def cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("this test needs a CUDA device (run with -m 'not gpu' on a CPU box)")
    return torch
