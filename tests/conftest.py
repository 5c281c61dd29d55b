import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


def pytest_terminal_summary(terminalreporter):
    """Used fraction of the tolerance for every GPU-vs-oracle comparison (tests/gpu_util.assert_close)."""
    try:
        import gpu_util
    except Exception:
        return
    rows = gpu_util.MARGINS
    if not rows:
        return
    worst = {}
    for name, dtype, used, nerr, n in rows:
        k = (name, dtype)
        if k not in worst or used > worst[k][0]:
            worst[k] = (used, nerr, n)
    tr = terminalreporter
    tr.write_line("")
    tr.write_line("parity margins: max |gpu - ref| / (atol + rtol*|ref| [+ derived extra]) per tensor (1.0 = at the bound)")
    for (name, dtype), (used, nerr, n) in sorted(worst.items(), key=lambda kv: -kv[1][0])[:60]:
        tr.write_line(f"  {used:7.4f}  max|err|/max|ref| {nerr:9.3e}  n={n:<10d} {dtype:4s} {name}")
    if gpu_util.BUDGET_USE:
        tr.write_line("fp32 rounding budget (DESIGN.md §6.4): elements outside the stated bound and the largest (excess / budget)")
        for name, use, n_over, n in gpu_util.BUDGET_USE:
            tr.write_line(f"  excess/budget {use:7.4f}  outside stated bound {n_over:8d} of {n:<10d} {name}")
