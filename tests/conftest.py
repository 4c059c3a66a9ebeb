import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import wveg_oracle
    wveg_oracle.lib()
    return wveg_oracle


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The CUDA library is built in-tree (nvcc cross-compiles without a GPU); a no-op when it is up to date.
    There is no fallback: if it cannot be built the tests that need it fail."""
    from paper_2607_01164_b200 import build
    try:
        build.build()
    except Exception as e:  # pragma: no cover
        print(f"warning: could not build libgs.so: {e}", file=sys.stderr)
