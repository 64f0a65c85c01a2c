import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def small_grid():
    """BASELINE configs[0] grid: 19 zenith x 73 azimuth x 41 freq."""
    import aera_inputs as ai
    return ai.WORKLOADS[0].grid


@pytest.fixture(scope="session")
def small_table(small_grid):
    import aera_inputs as ai
    return ai.pattern_table(small_grid, "complex64")
