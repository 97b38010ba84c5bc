import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running full-size parity case")


def relerr(a, b):
    """DESIGN.md error metric: max|a-b| / max|b| over all cells; if max|b| = 0 require a == 0."""
    import numpy as np
    mb = float(np.abs(b).max())
    ma = float(np.abs(a - b).max())
    if mb == 0.0:
        return 0.0 if ma == 0.0 else float("inf")
    return ma / mb
