import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "sanitizer: runs a tiny case under compute-sanitizer (one tool per gpurun call; run explicitly)")


def pytest_collection_modifyitems(config, items):
    # `sanitizer` cases run only when asked for by name (-m sanitizer): one compute-sanitizer tool per gpurun call
    if "sanitizer" not in (config.getoption("-m") or ""):
        drop = [it for it in items if "sanitizer" in it.keywords]
        if drop:
            items[:] = [it for it in items if "sanitizer" not in it.keywords]
            config.hook.pytest_deselected(items=drop)
    import torch
    if torch.cuda.is_available():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords or "sanitizer" in it.keywords:
            it.add_marker(skip)


GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


def pytest_sessionstart(session):
    """Make sure both shared libraries exist (cheap when up to date): the gcc-built oracle and the
    nvcc-built CUDA library.  Building is not using: no test computes through a missing library."""
    import oracle
    from paper_2605_22698_b200 import build as lib_build
    oracle.build()
    lib_build.build()
