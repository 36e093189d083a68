import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


@pytest.fixture(params=[0, 1, 2, 4], ids=lambda s: f"S{s}")
def super_tile(request):
    """GPU parity must hold for every super-tile size of the single-pass encoder (0 = automatic)."""
    import paper_2601_05531_b200 as dn
    old = dn.SUPER_TILE
    dn.SUPER_TILE = request.param
    yield request.param
    dn.SUPER_TILE = old
