import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    # make sure libuep.so matches the sources (no-op when it is up to date; nvcc cross-compiles
    # without a GPU).  A failure here is not hidden: the ABI / parity tests then fail loudly.
    try:
        from paper_2606_04101_b200 import build as uep_build
        uep_build.build()
    except Exception as e:                                   # pragma: no cover
        print(f"[conftest] libuep build failed: {e}", file=sys.stderr)


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
