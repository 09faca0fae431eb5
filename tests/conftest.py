"""pytest configuration: the `gpu` marker separates B200 parity tests from the CPU suite.

    python -m pytest tests -q -m "not gpu"   # oracle pins, host logic, C-ABI symbols (no GPU needed)
    python -m pytest tests -q -m gpu         # CUDA path vs oracle, through the C-ABI, on a B200
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); calls the CUDA path through the C-ABI")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        have = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        have = False
    if have:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
