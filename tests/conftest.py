import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def _has_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    """`-m gpu` on a box without CUDA is an error of selection, not a silent pass: fail the session.  A plain run
    (no -m, or -m "not gpu") on such a box skips the gpu-marked tests."""
    if _has_cuda():
        return
    expr = (config.getoption("-m") or "").strip()
    if "gpu" in expr and "not gpu" not in expr:
        raise pytest.UsageError("-m gpu was requested but no CUDA device is available: the parity tests cannot run "
                                "here (there is no CPU fallback); run them on the B200 box")
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
