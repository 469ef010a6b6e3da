import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running CPU statistical test")


@pytest.fixture(scope="session")
def repo_root():
    return ROOT


@pytest.fixture(scope="session", autouse=True)
def _library_built():
    """The in-tree CUDA library is a build artefact (git-ignored): compile it once if it is not there.  A missing
    nvcc or a compile error fails the session loudly -- there is no CPU fallback to fall back to."""
    from paper_1804_03310_b200 import build as b
    if not os.path.exists(b.LIB):
        b.build()
