import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def built_library():
    """the in-tree C-ABI library is a build product (git-ignored): compile it when it is not there yet
    (nvcc cross-compiles without a GPU).  Nothing is substituted for it: a failed build fails the tests.
    Only the tests that load it ask for it (the GPU tests and tests/test_abi.py), so the oracle pins
    run on a machine without nvcc."""
    from paper_2010_11751_b200 import build
    return build.build()


def pytest_collection_modifyitems(config, items):
    for item in items:
        if item.get_closest_marker("gpu") or item.module.__name__.endswith("test_abi"):
            if "built_library" not in item.fixturenames:
                item.fixturenames.insert(0, "built_library")


@pytest.fixture(scope="session")
def oracle():
    from oracle import lbm_oracle
    lbm_oracle.lib()
    return lbm_oracle
