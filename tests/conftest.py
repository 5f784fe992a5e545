import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "oracle"))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size configs (tens of seconds of oracle time)")


@pytest.fixture(scope="session")
def oracle():
    import ddhf_oracle
    ddhf_oracle.lib()
    return ddhf_oracle


@pytest.fixture(scope="session", autouse=True)
def _built_cuda_library():
    """libddhf.so is built in-tree by nvcc and is not in the git history: build it if it is missing
    or older than its sources (a no-op otherwise).  The product itself never builds or falls back:
    binding.lib() raises when the library is absent."""
    from paper_2603_08386_b200 import build
    build.build()
