import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def grid1():
    from paper_2009_06635_b200 import workloads as W
    return W.grid_config1()


@pytest.fixture(scope="session")
def grid2():
    from paper_2009_06635_b200 import workloads as W
    return W.grid_nnpdf_shaped()


@pytest.fixture(scope="session")
def ograph1(grid1):
    import oracle
    return oracle.OraclePdfGrid.from_spec(grid1)


@pytest.fixture(scope="session")
def ograph2(grid2):
    import oracle
    return oracle.OraclePdfGrid.from_spec(grid2)
