import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tiny_system():
    import nolsm_inputs as gi
    return gi.make_water_system(32, 6.0)


@pytest.fixture(scope="session")
def tiny_solution(tiny_system):
    import oracle.nolsm_oracle as orc
    return orc.solve_system(tiny_system)


@pytest.fixture(scope="session")
def mid_system_cpu():
    import nolsm_inputs as gi
    return gi.make_water_system(216, 8.0)
