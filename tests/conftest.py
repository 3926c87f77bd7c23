import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


def pytest_terminal_summary(terminalreporter):
    """Parity bookkeeping (tests/parity_util.py): how many configurations each check compared and how many of them
    used the conditioning exception of DESIGN.md §4.  Printed under -q as well."""
    try:
        import parity_util
    except Exception:
        return
    st = parity_util.STATS
    if not st:
        return
    tr = terminalreporter
    used = [s for s in st if s["exceptions"]]
    tr.write_line(f"parity: {len(st)} checks, {sum(s['batch'] for s in st)} configurations compared with the oracle, "
                  f"{sum(s['exceptions'] for s in st)} conditioning exceptions in {len(used)} checks; "
                  f"max strict rel err {max(s['max_rel_strict'] for s in st):.2e}")
    for s in used:
        tr.write_line(f"  parity exception: {s['label'] or '?'} n={s['n']} {s['which']}: {s['exceptions']}/{s['batch']} "
                      f"(worst {s['worst_exception_sigmas']:.2f} sigma of the FP64 relabelling scatter)")
