import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box via gpurun)")
    # Build step, not a fallback: if the in-tree CUDA library is missing or older than its sources and nvcc is here,
    # compile it (sm_100a cross-compiles without a GPU).  Without nvcc the import of the binding fails loudly.
    import shutil
    if shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc"):
        from paper_2606_17107_b200 import build as kbuild
        kbuild.build()


@pytest.fixture(scope="session")
def oracle():
    from oracle import kvr_oracle
    kvr_oracle.lib()
    return kvr_oracle
