"""pytest configuration: the `gpu` marker and shared seeded fixtures.

`-m "not gpu"` tests pin the CPU oracle (oracle/) against theory and check host-side logic;
`-m gpu` tests compare the CUDA path with the oracle through the C-ABI (libbq.so).
"""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def relmax(a, b):
    """max_i |a_i - b_i| / max_i |b_i| over real components (SURVEY.md §8(c) acceptance (i))."""
    a = np.asarray(a)
    b = np.asarray(b)
    d = np.abs(np.concatenate([(a - b).real.ravel(), (a - b).imag.ravel()])).max()
    n = np.abs(np.concatenate([b.real.ravel(), b.imag.ravel()])).max()
    return d / n


@pytest.fixture(scope="session")
def cfg1():
    """BASELINE.json config 1: 4^4, eps = 0.3, kappa = 0.12, antiperiodic t."""
    from paper_2111_04457_b200 import inputs
    L = (4, 4, 4, 4)
    seed = inputs.BASE_SEED + 1
    return dict(L=L, seed=seed, kappa=0.12, U=inputs.gauge(L, seed, 0.3), b=inputs.spinor(L, seed))
