import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def O():
    """The fp64 CPU oracle (test infrastructure)."""
    from oracle import sph_oracle
    sph_oracle.build()
    return sph_oracle


@pytest.fixture(scope="session")
def WL():
    from paper_1909_04504_b200 import workloads
    return workloads


def golden_path(name: str) -> str:
    return os.path.join(ROOT, "tests", "golden", name)
