import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def W():
    from paper_1809_02532_b200 import workloads
    return workloads


def random_state(rng, n, mass_ratio=25.0, vel=0.3):
    """A generic physical state: positive densities and temperatures, O(1) fields."""
    P = rng.uniform(-1.0, 1.0, size=(n, 18))
    P[:, 8] = rng.uniform(0.5, 1.5, n)
    P[:, 9] = rng.uniform(0.5, 1.5, n) / mass_ratio
    P[:, 10:16] = rng.uniform(-vel, vel, size=(n, 6))
    P[:, 16] = rng.uniform(0.3, 0.8, n)
    P[:, 17] = rng.uniform(0.3, 0.8, n)
    return P


def rot18(theta):
    """18x18 matrix rotating the in-plane components of B, E, u_i, u_e by theta."""
    c, s = np.cos(theta), np.sin(theta)
    Q = np.eye(18)
    for b in (0, 3, 10, 13):
        Q[b:b + 2, b:b + 2] = [[c, -s], [s, c]]
    return Q
