import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def _has_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if _has_cuda():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


def pytest_sessionstart(session):
    """The C-ABI library is built in-tree and is not in git: (re)build it when it is missing or older than its
    sources (nvcc cross-compiles without a GPU).  A failed build is left to the tests to report - they raise when the
    library is missing; nothing falls back to a CPU path."""
    try:
        from paper_1712_09434_b200.build import build
        build()
    except Exception as e:  # noqa: BLE001
        sys.stderr.write(f"conftest: building libtpc_tracker.so failed: {e}\n")
