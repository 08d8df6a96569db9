import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def pytest_sessionstart(session):
    """Build libchfsi.so if it is missing or older than its sources (nvcc cross-compiles without a GPU).  This is the
    same CUDA library, not a fallback: the binding itself still refuses to load anything else."""
    try:
        from paper_2605_30128_b200 import build
        build.build()
    except Exception as e:                                  # no nvcc here: the tests that need the library will say so
        print(f"conftest: libchfsi.so not (re)built: {e}")
