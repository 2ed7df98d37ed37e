import os
import sys

import pytest

# The oracle (oracle/ba_oracle.c) uses OpenMP; on a box whose cores are shared, actively spinning idle threads
# make it many times slower.  Must be set before libgomp is loaded; it does not touch the oracle's arithmetic.
os.environ.setdefault("OMP_WAIT_POLICY", "passive")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")
    config.addinivalue_line("markers", "slow: long-running case")


def pytest_collection_modifyitems(config, items):
    # GPU tests must fail loudly, not skip, when selected with -m gpu on a box without CUDA;
    # but a plain `pytest tests/` on a CPU box should not try them.
    try:
        import torch
        has_cuda = torch.cuda.is_available()
    except Exception:
        has_cuda = False
    markexpr = config.getoption("-m") or ""
    if has_cuda or "gpu" in markexpr.replace("not gpu", ""):
        return
    skip = pytest.mark.skip(reason="no CUDA device; run with -m gpu on a B200")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
