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
def _library_built(request):
    """The in-tree CUDA library is a build artefact (git-ignored): compile it once if it is not there.  Only the tests
    that load it need it (the `gpu` ones and tests/test_abi.py): when none of those is selected -- an oracle-only run on a box
    without nvcc -- nothing is built; otherwise a missing nvcc or a compile error fails the session loudly (there is
    no CPU fallback to fall back to)."""
    need = any(it.get_closest_marker("gpu") is not None or it.fspath.basename in ("test_abi.py",) for it in request.session.items)
    if not need:
        return
    from paper_1804_03310_b200 import build as b
    if not os.path.exists(b.LIB):
        b.build()
