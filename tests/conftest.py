import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: longer oracle runs")


@pytest.fixture(scope="session")
def ncpu():
    return max(1, min(8, os.cpu_count() or 1))


def pytest_terminal_summary(terminalreporter):
    """fp32 whole-run parity: the strict per-variable S14 error beside the norm actually asserted (S14 or S14')."""
    try:
        from util import FP32_LOG
    except Exception:
        return
    if not FP32_LOG:
        return
    worst = {}
    for label, v, strict, norm, e in FP32_LOG:
        k = (label, v, norm)
        if k not in worst or e > worst[k][1]:
            worst[k] = (strict, e)
    tr = terminalreporter
    tr.write_line("fp32 parity norms (label, variable, norm asserted: error; strict per-variable S14 error):")
    for (label, v, norm), (strict, e) in sorted(worst.items()):
        if norm == "S14'" or strict > 2e-6:
            tr.write_line("  %-34s var %d  %-4s %.2e   strict %.2e" % (label, v, norm, e, strict))
