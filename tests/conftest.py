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
    from oracle.oracle import Oracle
    return Oracle()


@pytest.fixture(scope="session")
def oracle_lso():
    """the oracle reading parameter rows as the state at plunge (reading D12): a separate instance, so that the
    forward-anchored `oracle` is never switched"""
    from oracle.oracle import Oracle
    return Oracle(anchor=True)


@pytest.fixture(scope="session")
def oracle_ld():
    from oracle.oracle import Oracle
    return Oracle(long_double=True)
