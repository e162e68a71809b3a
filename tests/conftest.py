import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def po():
    """The CPU oracle's ctypes driver (builds oracle/libmpm_oracle.so with gcc on first use)."""
    from oracle import pyoracle
    pyoracle._load()
    return pyoracle


@pytest.fixture(scope="session")
def mpm():
    """The CUDA path's binding; fails loudly when the library or a GPU is missing."""
    from paper_2404_17057_b200 import binding
    binding.load()
    return binding
