import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def W():
    from paper_2007_03678_b200 import workloads
    return workloads


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def par(orc, W):
    return orc.params(W.DEFAULT_PARAMS)


@pytest.fixture(scope="session")
def tiny(W, orc):
    grids, lig = W.make_config("tiny")
    return dict(grids=grids, lig=lig, og=orc.Grids.from_workload(grids), ol=orc.Ligand.from_workload(lig))


@pytest.fixture(scope="session")
def mid(W, orc):
    """drug-like ligand (40 atoms, 8 torsions, 7 types) on a reduced 32^3 grid: CPU-sized."""
    grids, lig = W.make_config("drug", grid_n=32)
    return dict(grids=grids, lig=lig, og=orc.Grids.from_workload(grids), ol=orc.Ligand.from_workload(lig))
