import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def c1():
    """BASELINE.json configs[0] (C1): one sector, 200 tracks, 5 % noise, seed 1."""
    from paper_2601_20569_b200 import datagen as dg
    return dg.generate(dg.preset("C1"))


@pytest.fixture(scope="session")
def c1_oracle(c1):
    import oracle
    return oracle.run(c1[0])
