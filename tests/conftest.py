import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def qdp():
    """The CUDA path's Python binding; only -m gpu tests and the symbol test use it."""
    from paper_1111_5596_b200.build import LIB, build
    if not os.path.exists(LIB):      # fresh checkout: the .so is a build artefact, not in the history
        build()
    import paper_1111_5596_b200 as q
    return q
