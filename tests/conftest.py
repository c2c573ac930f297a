import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def random_states(n, seed, r_scale=(8.0, 40.0), p_scale=(0.1, 0.35)):
    """Generic random phase-space points (not a workload): r, p isotropic, unit spins."""
    rng = np.random.default_rng(seed)

    def iso(k):
        v = rng.normal(size=(3, k))
        return v / np.linalg.norm(v, axis=0)

    z = np.zeros((12, n))
    z[0:3] = iso(n) * rng.uniform(*r_scale, n)
    z[3:6] = iso(n) * rng.uniform(*p_scale, n)
    z[6:9] = iso(n)
    z[9:12] = iso(n)
    return z


@pytest.fixture
def rand_states():
    return random_states
