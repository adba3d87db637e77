import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _ensure_built():
    """The .so files are build artefacts (git-ignored): (re)build them in-tree when missing or stale so that
    a fresh checkout can run the suite (nvcc cross-compiles sm_100a without a GPU; gcc for the oracle)."""
    try:
        from paper_1501_03869_b200 import build as pb
        pb.build()
    except Exception as e:                      # the ABI tests then fail loudly with the real reason
        print("WARNING: could not build libpat_b200.so: %s" % e)
    try:
        from oracle import build as ob
        ob.build()
    except Exception as e:
        print("WARNING: could not build the oracle: %s" % e)


def pytest_configure(config):
    _ensure_built()
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: long-running full-size case")


def _has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if _has_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
