import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def tiny_inputs():
    from paper_2410_09189_b200.workloads import WORKLOADS, make_inputs_numpy
    w = WORKLOADS["tiny"]
    Phi, eps, occ = make_inputs_numpy(w)
    return w, Phi, eps, occ
