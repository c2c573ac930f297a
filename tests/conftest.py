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


def config3_sample():
    """The cells of BASELINE config 3 that the full-length class tests recompute with the oracle: 400 drawn uniformly from
    the 314 x 314 grid (north_star's bar is on grid cells) + 100 more from the strong-field rows r0 < 18, where every
    chaotic and dropped cell lives.  Returns (global cell indices, mask of the uniform part)."""
    rng = np.random.default_rng(8)
    uni = rng.choice(314 * 314, 400, replace=False)
    strong = np.setdiff1d(rng.choice(314 * 50, 110, replace=False), uni)[:100]
    idx = np.concatenate([uni, strong])
    return idx, np.arange(idx.size) < uni.size
