import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    # The product never builds itself (hydro.lib() fails loudly without libgamer_hydro.so); the TEST SESSION may: a fresh
    # checkout has no binaries, nvcc cross-compiles without a device, and build() is a no-op when the library is newer
    # than its sources.
    from paper_0907_3390_b200 import build as cuda_build
    cuda_build.build()
    from oracle import build as oracle_build       # the checker too, before any test starts worker processes
    oracle_build.build()


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
