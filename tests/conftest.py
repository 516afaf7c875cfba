import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session", autouse=True)
def _libpm_built():
    """Build libpm.so (and the generated kernels) if it is missing or older than its sources: an explicit build step,
    not a fallback — the library itself still refuses to run without its CUDA extension."""
    from paper_1508_07441_b200.csrc import build
    build.build()


@pytest.fixture(scope="session")
def oracle():
    from oracle.pm_oracle import Oracle
    return Oracle()


@pytest.fixture(scope="session")
def oracle_ld():
    from oracle.pm_oracle import Oracle
    return Oracle(long_double=True)
