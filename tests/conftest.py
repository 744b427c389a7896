import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HERE = os.path.dirname(os.path.abspath(__file__))
for _p in (HERE, ROOT):          # ROOT first on sys.path; HERE for `import parity_util`
    if _p not in sys.path:
        sys.path.insert(0, _p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (run with -m gpu on the GPU box)")


def pytest_terminal_summary(terminalreporter):
    """Every loss comparison of the GPU parity tests: how ill-conditioned the sum was and whether
    north_star's 1e-5 relative bar alone (without DESIGN.md's conditioning floor) passed."""
    try:
        import parity_util as P
    except Exception:
        return
    if not P.LOSS_LOG:
        return
    n = len(P.LOSS_LOG)
    rel_ok = sum(1 for e in P.LOSS_LOG if e[5])
    tr = terminalreporter
    tr.write_line("loss parity: %d comparisons, %d within 1e-5 |loss| alone, %d needed the "
                  "1e-6 sum|term| conditioning floor" % (n, rel_ok, n - rel_ok))
    for label, aloss, cond, diff, rel_tol, ok in P.LOSS_LOG:
        if not ok:
            tr.write_line("  floor needed: %-28s |loss| %.3e  sum|term|/|sum term| %.3e  |diff| %.3e "
                          "(1e-5 |loss| = %.3e)" % (label, aloss, cond, diff, rel_tol))
    conds = sorted(e[2] for e in P.LOSS_LOG if e[2] != float("inf"))
    if conds:
        tr.write_line("  conditioning sum|term|/|sum term|: min %.2f median %.2f max %.3e" % (
            conds[0], conds[len(conds) // 2], conds[-1]))
