"""pytest configuration: markers, import path, shared helpers."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: takes more than ~20 s")
    config.addinivalue_line("markers", "huge: needs > 100 GB of device memory (configs C4/C5 at full size)")


def rel_l2(a, b):
    """||a-b||_2 / ||b||_2 (b = oracle); north_star's first parity metric."""
    import numpy as np
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def max_rel_peak(a, b):
    """max|a-b| / max|b| (b = oracle); north_star's second parity metric."""
    import numpy as np
    a = np.asarray(a)
    b = np.asarray(b)
    return float(np.abs(a - b).max() / np.abs(b).max())
