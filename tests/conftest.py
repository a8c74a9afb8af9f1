import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def ref():
    from oracle import ref as _ref
    _ref.build()
    return _ref


@pytest.fixture(scope="session")
def mech9():
    from paper_2504_13750_b200 import inputs
    return inputs.synthetic_mechanism(9, 21)


@pytest.fixture(scope="session")
def mech20():
    from paper_2504_13750_b200 import inputs
    return inputs.synthetic_mechanism(20, 100)
