import os
import subprocess
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
    from oracle import build as oracle_build       # the checker, before any test starts worker processes: mandatory
    oracle_build.build()
    from paper_0907_3390_b200 import build as cuda_build
    try:
        cuda_build.build()
    except (FileNotFoundError, subprocess.CalledProcessError) as exc:
        # No nvcc on this machine, or a compile error.  The oracle-only tests (its pins, its multi-step loop) do not
        # need the CUDA library and still run; a test that reaches for the library is skipped on a machine without a
        # GPU and FAILS on a machine with one (a GPU box that cannot build the product must not look green).
        _library_unavailable("libgamer_hydro.so could not be built: %r" % (exc,))


def _library_unavailable(reason):
    from paper_0907_3390_b200 import hydro

    def lib():
        try:
            import torch
            has_gpu = torch.cuda.is_available()
        except Exception:
            has_gpu = False
        if has_gpu:
            raise ImportError(reason + " (there is no CPU fallback)")
        pytest.skip(reason)

    hydro._lib = None
    hydro.lib = lib


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
