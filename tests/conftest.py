import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle64():
    import oracle
    return oracle.Oracle("f64")


@pytest.fixture(scope="session")
def oracle80():
    import oracle
    return oracle.Oracle("f80")


@pytest.fixture(scope="session")
def oracleC():
    """REAL = long double _Complex build: exact Jacobian action by complex-step differentiation."""
    import oracle
    return oracle.Oracle("c80")
