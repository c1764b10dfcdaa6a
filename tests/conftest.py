import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (sm_100a); run with -m gpu on the B200 box")
    config.addinivalue_line("markers", "slow: long-running full-size case")


def pytest_collection_modifyitems(config, items):
    # A gpu-marked test must fail loudly, not skip silently, when selected on a box without a GPU.
    pass


@pytest.fixture(scope="session")
def _built_library():
    """Build libmfsdp.so in-tree if it is missing or stale (nvcc cross-compiles without a GPU)."""
    from paper_2607_05895_b200 import build as _build
    _build.build()


@pytest.fixture(autouse=True)
def _library_for_product_tests(request):
    """Every test except the oracle pins (tests/test_oracle_*.py) needs the built library; the pins must run on a box
    without nvcc, so they do not depend on the product building."""
    if not os.path.basename(str(request.node.fspath)).startswith("test_oracle_"):
        request.getfixturevalue("_built_library")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")
