import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc_ld():
    import oracle
    return oracle.Oracle("ld")


@pytest.fixture(scope="session")
def orc_q():
    import oracle
    return oracle.Oracle("q")


@pytest.fixture(scope="session")
def orc_f64():
    import oracle
    return oracle.Oracle("f64")
