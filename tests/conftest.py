"""Shared fixtures.  `-m "not gpu"` tests run on a CPU-only box; `-m gpu` tests need a B200."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


_GRID_CACHE = {}


def oracle_grid(level, smooth=True):
    """Grid from the ORACLE's own generator (never from the CUDA library), cached per session."""
    from oracle import grid_oracle
    key = (level, smooth)
    if key not in _GRID_CACHE:
        xyz, nbr, C, _ = grid_oracle.build(level, smooth=smooth, tol=1e-8)
        _GRID_CACHE[key] = (xyz, nbr, C)
    return _GRID_CACHE[key]


@pytest.fixture(scope="session")
def ogrid():
    return oracle_grid


def have_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False
