import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def inputs():
    from paper_2601_14301_b200 import inputs as m
    return m


@pytest.fixture(scope="session")
def cfg1(inputs):
    return inputs.WORKLOADS["cfg1"]


@pytest.fixture(scope="session")
def oracle_cfg1(inputs, cfg1):
    import oracle
    return oracle.from_workload(cfg1, inputs)
