"""pytest configuration: the `gpu` marker and repo-root imports.

`-m "not gpu"` : oracle pins, input generator, host logic, C-ABI symbol checks (CPU only).
`-m gpu`       : parity tests proper -- CUDA path vs oracle through the C-ABI (needs a B200).
"""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


def pytest_collection_modifyitems(config, items):
    # GPU tests are skipped (not failed) on a box without a device, so a plain
    # `pytest tests/` works here; `-m gpu` on the GPU box runs them all.
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
