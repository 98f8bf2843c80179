import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def rel_l2(a, b):
    import numpy as np
    a = np.asarray(a)
    b = np.asarray(b)
    den = np.sqrt(np.sum(np.abs(b) ** 2))
    num = np.sqrt(np.sum(np.abs(a - b) ** 2))
    return float(num / den) if den > 0 else float(num)


@pytest.fixture(scope="session")
def small_plan_args():
    # fs, N, Q, fmin, fmax, rows : a 256-sample plan whose rows span several M buckets
    return dict(fs=256.0, N=256, Q=[4.0, 8.0], fmin=8.0, fmax=100.0, spacing=7)
