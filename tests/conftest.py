import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def c0():
    import gen
    return gen.make_problem(0)


@pytest.fixture(scope="session")
def c0_walkers(c0):
    import gen
    return gen.make_walkers(c0)


@pytest.fixture(scope="session")
def c1():
    import gen
    return gen.make_problem(1)


@pytest.fixture(scope="session")
def c1_walkers(c1):
    import gen
    return gen.make_walkers(c1, n_w=16)
