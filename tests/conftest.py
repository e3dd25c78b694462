import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def tiny():
    from paper_2412_08265_b200 import synth
    return synth.make_workload("tiny")


@pytest.fixture(scope="session")
def small():
    from paper_2412_08265_b200 import synth
    return synth.make_workload("small")


@pytest.fixture(scope="session")
def small_oracle_cube(small):
    """fp64 oracle cube of config 1 (about 2 s on 8 cores); shared by several tests."""
    import oracle
    return oracle.build_cube(small.particles, small.rotation, small.ssp, small.telescope)
