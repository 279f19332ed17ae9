import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


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


@pytest.fixture(scope="session", autouse=True)
def _native_libraries_are_built():
    """libecpush.so (nvcc, sm_100a) and liboracle.so (gcc) are built in-tree if missing or stale.  Building the
    product library is not a fallback: if nvcc fails the session fails."""
    from paper_2603_16624_b200 import build as product_build
    from oracle import build as oracle_build
    product_build.build()
    oracle_build.build()
