import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running full-size case")


def load_golden(name):
    """Parse tests/golden/<name>: '#' comments, 'key = v1 v2 ...' lines -> {key: [floats]}."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split("=", 1)
            out[k.strip()] = [float(x) for x in v.split()]
    return out


import contextlib
import ctypes


@contextlib.contextmanager
def omp_threads(n):
    """Run the oracle's OpenMP loops with n threads inside the block (tiny meshes stepped thousands of times spend
    their time in thread wake-ups otherwise); restores the default afterwards."""
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        old = gomp.omp_get_max_threads()
        gomp.omp_set_num_threads(int(n))
    except OSError:
        gomp = None
    try:
        yield
    finally:
        if gomp is not None:
            gomp.omp_set_num_threads(old)
