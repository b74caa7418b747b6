import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def _has_gpu() -> bool:
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if _has_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


# The parity tests print what they measured (worst |d|/RMS, rel L2, score differences).  pytest -q shows the output of
# failing tests only, so the lines of PASSING tests are collected here and printed as one section at the end of the run:
# the numbers behind "passed" are in the log whoever runs the suite.
_MEASURED = []


def pytest_runtest_logreport(report):
    if report.when != "call" or not report.passed:
        return
    for line in (report.capstdout or "").splitlines():
        if any(k in line for k in ("worst", "max |d|", "rel L2", "MISSES")):
            _MEASURED.append(f"{report.nodeid.split('::')[-1]}: {line.strip()}")


def pytest_terminal_summary(terminalreporter):
    if not _MEASURED:
        return
    terminalreporter.section("measured parity (CUDA path vs oracle)")
    for line in _MEASURED:
        terminalreporter.write_line(line[:400])
