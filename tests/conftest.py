import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    from oracle import oracle as O
    O.build()          # the checker is plain C; gcc builds it in a second


@pytest.fixture(scope="session")
def O():
    from oracle import oracle as orc
    return orc


@pytest.fixture(scope="session")
def W():
    from paper_2511_17701_b200 import workloads
    return workloads


def pytest_terminal_summary(terminalreporter):
    """Evidence for the two FP32 allowances of the parity rules, printed with every GPU run."""
    try:
        from oracle import parity as helpers
        rows = helpers.AXIS_STATS
    except Exception:
        return
    if not rows:
        return
    tr = terminalreporter
    for prec in ("f32", "f64"):
        r = [x for x in rows if x[0] == prec]
        if not r:
            continue
        n_ax = sum(x[2] for x in r)
        tr.write_line(f"[parity] {prec}: {len(r)} particle comparisons, {sum(x[1] for x in r)} particles; "
                      f"axis allowance (kappa > 1) used by {n_ax} particles in {sum(1 for x in r if x[2])} comparisons, "
                      f"their max raw error {max(x[3] for x in r):.2e} (tolerance {helpers.TOL[prec]['x']:.0e}), max kappa {max(x[4] for x in r):.1f}")
    try:
        s = helpers.STRADDLE_STEPS
        tr.write_line(f"[parity] steps whose J comparison substituted face-straddling particles: {len(s)} "
                      f"({sum(n for _, n in s)} particles; by precision: " +
                      ", ".join(f"{p} {sum(1 for q, _ in s if q == p)}" for p in ("f32", "f64")) + ")")
    except Exception:
        pass
