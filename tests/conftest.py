import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    """The CPU oracle (built on first use).  Test infrastructure only."""
    import oracle as _oracle
    _oracle._load()
    return _oracle


@pytest.fixture(scope="session")
def das_lib():
    """The CUDA product library through its Python binding; builds it if missing."""
    import paper_2606_13259_b200 as das
    das.load()
    return das
