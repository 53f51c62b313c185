import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    """The CPU oracle (test infrastructure), built on demand with gcc."""
    import oracle

    oracle.num_threads()
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The C-ABI library is built in-tree (nvcc cross-compiles without a GPU); a stale or missing libtpt.so is rebuilt
    once per session so that the GPU tests never run against an old binary.  Without nvcc the tests that need the
    library fail loudly in api.lib() (there is no fallback)."""
    import shutil

    from paper_2603_09528_b200 import build

    if shutil.which("nvcc") or os.path.exists("/usr/local/cuda/bin/nvcc"):
        build.build()
    yield
