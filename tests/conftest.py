import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on a B200 with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    """The CPU oracle (built on demand with g++).  Test infrastructure only."""
    from oracle import pt_oracle
    pt_oracle.build()
    return pt_oracle


@pytest.fixture(scope="session")
def golden_basis():
    import numpy as np
    path = os.path.join(ROOT, "tests", "golden", "ma_basis_definition.txt")
    rows = [ln.split() for ln in open(path) if not ln.startswith("#")]
    return np.array([[float(x) for x in r] for r in rows])


@pytest.fixture(scope="session")
def golden_config1():
    import numpy as np
    path = os.path.join(ROOT, "tests", "golden", "config1_worked.txt")
    rows = [ln.split() for ln in open(path) if not ln.startswith("#")]
    return np.array([[float(x) for x in r] for r in rows])
