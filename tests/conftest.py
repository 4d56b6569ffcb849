import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


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


def pytest_sessionfinish(session, exitstatus):
    """With OSIV_CHECK_BUILD=1 the whole GPU suite runs on the library built with device-side index checks
    (include/osiv.h: osiv_debug_checks); any out-of-range gather index seen during the session fails it here."""
    if os.environ.get("OSIV_CHECK_BUILD", "") != "1":
        return
    try:
        import paper_1903_10088_b200 as osiv
        r = osiv.debug_checks()
    except Exception as e:                      # the library was never loaded (CPU-only session)
        print(f"\nindex checks: not available ({e})")
        return
    print(f"\nindex checks (OSIV_CHECK_BUILD=1): {r}")
    if r["violations"] != 0:
        session.exitstatus = 1
