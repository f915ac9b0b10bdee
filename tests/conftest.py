import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    """Tests marked gpu are skipped when no device is visible -- unless the run asked for them (`-m gpu`): then a
    missing device is an error, not a green run with nothing executed."""
    try:
        import torch
        has = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has = False
    if has:
        return
    asked = (config.getoption("-m") or "").strip()
    if asked == "gpu" and any("gpu" in it.keywords for it in items):
        raise pytest.UsageError("-m gpu was requested but no CUDA device is visible")
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)
