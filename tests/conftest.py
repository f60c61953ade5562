import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def cfg1():
    from paper_2603_21835_b200 import workloads
    return workloads.make("si8_sz")


@pytest.fixture(scope="session")
def cfg1_oracle(cfg1):
    import oracle
    w = cfg1
    H, blocks = oracle.vlocal(w.lattice, w.ngrid, w.species, w.atom_species, w.atom_pos, w.V)
    return H, blocks
