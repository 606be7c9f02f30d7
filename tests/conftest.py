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
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


def pytest_terminal_summary(terminalreporter, exitstatus, config):
    """north_star: "any near-threshold ties are logged": the parity harness' tie log is written to
    gpurun_out/ties.json (the folder that comes back from a GPU run) and its size is printed here."""
    parity = sys.modules.get("parity")
    if parity is None:
        return
    try:
        import torch
        if not torch.cuda.is_available():
            return          # the CPU suite compares nothing with the CUDA path: it leaves a GPU run's log alone
    except Exception:
        return
    path = os.path.join(ROOT, "gpurun_out", "ties.json")
    try:
        kinds = parity.dump_ties(path)
    except OSError as e:
        terminalreporter.write_line(f"parity ties: {len(parity.TIES)} (not written: {e})")
        return
    terminalreporter.write_line(f"parity ties logged: {len(parity.TIES)} {kinds} -> {path}")
