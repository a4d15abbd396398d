import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """the in-tree C-ABI library is a build product (git-ignored): compile it when it is not there yet
    (nvcc cross-compiles without a GPU).  Nothing is substituted for it: a failed build fails the tests."""
    from paper_2010_11751_b200 import build
    build.build()


@pytest.fixture(scope="session")
def oracle():
    from oracle import lbm_oracle
    lbm_oracle.lib()
    return lbm_oracle
