import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "oracle")):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def po():
    """The CPU oracle (test infrastructure)."""
    import pyoracle

    pyoracle.lib()
    return pyoracle


@pytest.fixture(scope="session")
def W():
    from paper_2006_07964_b200 import workloads

    return workloads
