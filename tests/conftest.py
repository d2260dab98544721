import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _libmss_present():
    """libmss.so is built in-tree (python -m paper_1403_2136_b200.build / __graft_entry__.build()); if a checkout has none
    yet and nvcc is at hand, build it once so that the ABI and GPU tests exercise the CUDA path (there is no fallback)."""
    import shutil
    from paper_1403_2136_b200 import binding, build as mss_build
    if not os.path.exists(binding.lib_path()) and (shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc")):
        mss_build.build()
    yield
