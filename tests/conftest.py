import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def f32_to_bf16_bits(x):
    """Round-to-nearest-even float -> bf16 bit patterns (uint16).  Test helper."""
    u = np.ascontiguousarray(x, np.float32).view(np.uint32).astype(np.uint64)
    u = u + 0x7FFF + ((u >> 16) & 1)
    return (u >> 16).astype(np.uint16)


def randn_bf16(rng, *shape):
    return f32_to_bf16_bits(rng.standard_normal(shape).astype(np.float32))


@pytest.fixture
def nprng():
    return np.random.default_rng(20250221)
