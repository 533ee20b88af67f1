import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def make_oracle(L, L5, M5, b5, c5, mf, eps, seed):
    """Oracle instance on the seeded synthetic gauge field of paper_1701_07559_b200.inputs."""
    from oracle.mdwf_oracle import MdwfOracle
    from paper_1701_07559_b200 import inputs
    U = inputs.gauge_field(L, eps, seed).numpy()
    return MdwfOracle(L, L5, M5, b5, c5, mf, U)


def gaussian(orc, seed):
    from paper_1701_07559_b200 import inputs
    return inputs.gaussian_source(orc.L, orc.L5, seed).numpy()


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


@pytest.fixture(scope="session")
def orc_cfg1():
    """configs[0] of BASELINE.json: 4^4, L5=8, M5=1.3, b5=1.5, c5=0.5, m_f=0.05, eps=0.3, seed 0."""
    return make_oracle((4, 4, 4, 4), 8, 1.3, 1.5, 0.5, 0.05, 0.3, 0)


@pytest.fixture(scope="session")
def orc_ragged():
    """distinct extents 4x2x2x6 (index-order bugs), b5 - c5 != 1."""
    return make_oracle((4, 2, 2, 6), 4, 1.2, 1.4, 0.7, 0.03, 0.4, 11)
