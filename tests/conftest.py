import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_sessionstart(session):
    """Build the C-ABI CUDA library in-tree if it is missing or older than its sources (nvcc cross-compiles without a
    GPU); the oracle builds itself on first use.  A failing build fails the session loudly: there is no fallback."""
    from paper_2607_06337_b200 import build as ob_build
    ob_build.build()


def pytest_collection_modifyitems(config, items):
    """GPU tests are skipped (not failed) on a machine without a device."""
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


def pytest_terminal_summary(terminalreporter):
    """Worst per-element errors of the parity comparisons, per test (tests/helpers.py: rel_state_error)."""
    try:
        from helpers import WORST_PER_ELEMENT
    except Exception:  # pragma: no cover
        return
    if WORST_PER_ELEMENT:
        terminalreporter.write_line("per-element parity errors (A27 block norm | worst element vs block max | vs its own size):")
        for k, v in sorted(WORST_PER_ELEMENT.items()):
            terminalreporter.write_line(f"  {v['max']:.1e} | {v['max_inf']:.1e} | {v['max_own']:.1e}  {k}")
