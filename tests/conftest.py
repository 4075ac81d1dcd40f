import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_sessionstart(session):
    # Build the in-tree libraries if they are missing or older than their sources (a fresh checkout has no .so: they are
    # git-ignored).  A failure is reported once here and then loudly by every test that needs the library.
    try:
        import __graft_entry__
        __graft_entry__.build()
    except Exception as e:  # noqa: BLE001
        sys.stderr.write("conftest: building the libraries failed: %r\n" % (e,))


def pytest_collection_modifyitems(config, items):
    # A GPU test on a box without a GPU is an error in how the suite was invoked, not a skip:
    # the product has no CPU fallback.  Only auto-skip when the user did not ask for gpu tests.
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    markexpr = config.getoption("-m") or ""
    if "gpu" in markexpr and "not gpu" not in markexpr:
        return
    skip = pytest.mark.skip(reason="no CUDA device here; run with -m gpu on the GPU box")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
