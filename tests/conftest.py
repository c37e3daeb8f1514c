import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")


@pytest.fixture(scope="session")
def oracle():
    """The CPU oracle (oracle/niv_oracle.c through its ctypes wrapper), built on demand with gcc."""
    from oracle import niv_oracle
    niv_oracle.build()
    return niv_oracle
