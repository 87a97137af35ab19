import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HERE = os.path.dirname(os.path.abspath(__file__))
for _p in (ROOT, HERE):
    if _p not in sys.path:
        sys.path.insert(0, _p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); parity tests through the C ABI")
    config.addinivalue_line("markers", "slow: long-running oracle comparison")


@pytest.fixture(scope="session", autouse=True)
def _library_is_built():
    """libgh.so is built in-tree (nvcc cross-compiles without a GPU); a no-op when it is newer than its sources."""
    from paper_1804_09101_b200 import build

    build.build()


@pytest.fixture(scope="session")
def oracle():
    from oracle.gh_oracle import Oracle

    return Oracle("long double")


@pytest.fixture(scope="session")
def oracle_double():
    from oracle.gh_oracle import Oracle

    return Oracle("double")
