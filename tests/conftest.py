"""pytest configuration: markers, import path, session-cached workloads."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def normwise_rel_err(x: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """Per-Cartesian-component normwise relative error over the particle set:
    ||x[:,c] - ref[:,c]||_2 / ||ref[:,c]||_2."""
    x = np.asarray(x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    num = np.sqrt(((x - ref) ** 2).sum(axis=0))
    den = np.sqrt((ref ** 2).sum(axis=0))
    return num / den


_cache = {}


def workload(k: int, **kw):
    """Session-cached BASELINE.json configuration k (1..5)."""
    from paper_2210_02472_b200 import workloads as W
    key = (k, tuple(sorted(kw.items())))
    if key not in _cache:
        _cache[key] = W.CONFIGS[k](**kw)
    return _cache[key]
