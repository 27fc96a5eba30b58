import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")
    config.addinivalue_line("markers", "slow: large-config parity (minutes of oracle time)")


def pytest_collection_modifyitems(config, items):
    """GPU tests are skipped (not failed) where there is no device, e.g. a bare `pytest tests/`
    on the CPU box; `-m "not gpu"` deselects them anyway."""
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


def read_golden_sets(name):
    """Parse 'k1 k2 ... : m1 m2 ...' lines into (tuple(keys), frozenset(members))."""
    out = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            left, right = line.split(":")
            out.append((tuple(int(x) for x in left.split()), frozenset(int(x) for x in right.split())))
    return out
