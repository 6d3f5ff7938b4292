import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch

        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session", autouse=True)
def _native_code_built():
    """The CUDA library and the C oracle are built in-tree (git-ignored): make sure they exist
    and are not older than their sources.  A failed rebuild is tolerated only when a library is
    already there (e.g. a box without nvcc that received the built .so with the snapshot)."""
    from oracle import build_oracle
    from paper_2602_05255_b200 import build

    try:
        build.build()
    except Exception:
        if not os.path.exists(build.LIB):
            raise
    try:
        build_oracle.build()
    except Exception:
        pass      # tests that need the C oracle report its absence themselves
