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
    """Measured worst |a_gpu - a_ref| / S_i of the conditioning-aware rule (nf_testlib.assert_parity_conditioned)."""
    try:
        import nf_testlib
    except Exception:
        return
    if not nf_testlib.RATIOS:
        return
    worst = max(nf_testlib.RATIOS, key=lambda t: t[1])
    rows = sum(t[2] for t in nf_testlib.RATIOS)
    total = sum(t[3] for t in nf_testlib.RATIOS)
    tail = sum(t[4] for t in nf_testlib.RATIOS)
    tail_worst = max(nf_testlib.RATIOS, key=lambda t: t[5])
    terminalreporter.write_line(
        f"C13 rule: {len(nf_testlib.RATIOS)} comparisons, {total} rows; {rows} rows outside 1e-5 |a_ref| accepted by "
        f"C13 = {nf_testlib.C13:.1e} x S, worst err/S among them {worst[1]:.3e} [{worst[0]}]; {tail} rows "
        f"({100.0 * tail / max(total, 1):.4f} %) accepted by neither (the 0.1 % the rule allows), worst rel. error there "
        f"{tail_worst[5]:.3e} [{tail_worst[0]}]")
