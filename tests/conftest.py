import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg0():
    """BASELINE config 0: 3D 8^3 elements, bs 3 -> 6, 27 aggregates."""
    from paper_2606_24748_b200 import problems as pr
    g = pr.make_generator(0)
    g.build_prolongator(0)
    return g


@pytest.fixture(scope="session")
def grid2d():
    """A small 2D plane-strain grid (8x8 elements, bs 2 -> 3) for brute-force checks."""
    from paper_2606_24748_b200 import problems as pr
    g = pr.Generator(2, 8, seed=7)
    g.build_prolongator(0)
    return g
