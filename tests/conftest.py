import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_mod():
    """The CPU oracle (test infrastructure).  Compiles oracle/xy_oracle.cpp with g++ on first use."""
    from oracle import xy_oracle
    xy_oracle.lib()
    return xy_oracle


@pytest.fixture(scope="session")
def xy_mod():
    """The CUDA path.  Builds the C-ABI library in-tree if it is missing; never falls back."""
    import paper_1211_0780_b200 as pkg
    from paper_1211_0780_b200.build import build_library
    build_library()
    from paper_1211_0780_b200 import binding
    binding.load_library()
    return binding
