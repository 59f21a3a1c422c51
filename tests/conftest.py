import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


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


def _parity_totals():
    try:
        from tests.parity import PARITY_LOG
    except Exception:
        return None, []
    if not PARITY_LOG:
        return None, []
    tot = {k: sum(r[k] for r in PARITY_LOG) for k in ("problems", "excepted", "swapped_pages", "fp32_band_pages")}
    tot["max_rel"] = max(r["max_rel"] for r in PARITY_LOG)
    return tot, PARITY_LOG


def pytest_terminal_summary(terminalreporter):
    """How often the near-tie exception of the selection parity fired (visible under -q)."""
    tot, log = _parity_totals()
    if tot is None:
        return
    terminalreporter.write_line(
        f"selection parity: {tot['problems']} (request, head) problems checked against the oracle, near-tie rule used in "
        f"{tot['excepted']}, {tot['swapped_pages']} pages swapped (ceiling: {tot['fp32_band_pages']} oracle scores inside the "
        f"fp32 band), largest relative distance of a swapped page {tot['max_rel']:.2e}")
    out = os.path.join(ROOT, "gpurun_out")
    try:
        import json
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "parity_counts.json"), "w") as f:
            json.dump({"total": tot, "calls": log}, f, indent=1)
    except OSError:
        pass
