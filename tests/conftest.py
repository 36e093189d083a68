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


@pytest.fixture(params=[0, 1, 2, 4, "chained"], ids=lambda s: f"S{s}")
def super_tile(request):
    """GPU parity must hold for every super-tile size of the single-pass encoder (0 = automatic), with the regular-layout
    fast path in front of it (the default) and, in the "chained" variant, with the chained-scan encoder alone."""
    import paper_2601_05531_b200 as dn
    old, oldf = dn.SUPER_TILE, dn.FAST_PATH
    dn.SUPER_TILE = 0 if request.param == "chained" else request.param
    dn.FAST_PATH = 0 if request.param == "chained" else 2           # 2: the fast path on inputs of any size
    yield request.param
    dn.SUPER_TILE, dn.FAST_PATH = old, oldf
