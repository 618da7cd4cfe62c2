import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


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


# Lines the statistical parity tests want in the tail of the run whether they pass or not (how many shells needed
# the second look of DESIGN.md R21): collected in tests/parity_notes.py, printed after the last test.
def pytest_terminal_summary(terminalreporter):
    import parity_notes
    if parity_notes.NOTES:
        terminalreporter.section("T(r) parity: shells flagged on seeds 1-8 (DESIGN.md R21)")
        for line in parity_notes.NOTES:
            terminalreporter.write_line(line)
