import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def conformal():
    from paper_1802_04449_b200 import inputs
    return inputs.conformal_eos()


@pytest.fixture(scope="session")
def crossover():
    from paper_1802_04449_b200 import inputs
    return inputs.crossover_table()
