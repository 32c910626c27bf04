import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


def pytest_collection_modifyitems(config, items):
    """GPU tests must never pass silently on a box without a GPU."""
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:                                    # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


def pytest_terminal_summary(terminalreporter):
    """The relaxation of the 1-ulp bar made visible: totals of every element-wise bf16 comparison of the run."""
    mod = sys.modules.get("tests.parity")
    if mod is None or not mod.TOTALS["n"]:
        return
    t = mod.TOTALS
    terminalreporter.write_line(
        "bf16 parity (|g - bf16(o)| <= max(ulp, (m+4) 2^-24 S)): %d elements compared, %d bit-exact, %d within 1 ulp, "
        "%d needed the accumulation floor (%.2e of all), %d failed"
        % (t["n"], t["exact"], t["within_1ulp"], t["needed_floor"], t["needed_floor"] / t["n"], t["fail"]))
