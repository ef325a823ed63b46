"""pytest configuration: repo root on sys.path, `gpu` marker, shared helpers."""
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


def rng_uniform(seed, shape, lo=-1.0, hi=1.0):
    """Seeded uniform field from the workload module's splitmix64 (no solver arithmetic)."""
    from workloads import splitmix64_uniform

    n = int(np.prod(shape))
    return (lo + (hi - lo) * splitmix64_uniform(seed, n)).reshape(shape)


@pytest.fixture(scope="session")
def uniform():
    return rng_uniform
