import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")
    from parity_util import parity_log_path
    try:
        config._parity_log_start = os.path.getsize(parity_log_path())
    except OSError:
        config._parity_log_start = 0


def pytest_terminal_summary(terminalreporter, exitstatus, config):
    """What this run's parity checks needed beyond the 1e-12 / 1e-15 rule, test by test (from the parity
    log, tests/parity_util.py): a reader sees at once that the contract configs use no clause."""
    import json
    from parity_util import parity_log_path
    try:
        with open(parity_log_path()) as f:
            f.seek(getattr(config, "_parity_log_start", 0))
            recs = [json.loads(line) for line in f if line.strip()]
    except (OSError, ValueError):
        return
    if not recs:
        return
    tr = terminalreporter
    tr.section("parity summary")
    tr.write_line(f"{len(recs)} logged checks, {sum(r.get('n', 0) for r in recs)} outputs, "
                  f"max eq.1 difference {max(r.get('max_eq1', 0.0) for r in recs):.3e}")
    contract = [r for r in recs if r.get("what", "").startswith(("config", "alphas config"))]   # pdf_xfxq2 / alphas_q2 on configs 1-5
    tr.write_line(f"contract configs 1-5 (pdf_xfxq2, alphas_q2): {len(contract)} checks, {sum(r.get('n', 0) for r in contract)} outputs, "
                  f"n_clause = {sum(r.get('n_clause', 0) for r in contract)}")
    used = [r for r in recs if r.get("n_clause", 0) or r.get("n_slack", 0)]
    if not used:
        tr.write_line("no check used the conditioning clause or a coordinate allowance")
    for r in used:
        tr.write_line(f"  {r.get('what', '?')}: n = {r.get('n')}, clause uses = {r.get('n_clause', 0)} (max |d|/S = "
                      f"{r.get('max_d_over_S', 0.0):.3e}), t->1 allowance uses = {r.get('n_slack', 0)} "
                      f"(max |d|/allowance = {r.get('max_slack_used', 0.0):.2f})")


@pytest.fixture(scope="session")
def grid1():
    from paper_2009_06635_b200 import workloads as W
    return W.grid_config1()


@pytest.fixture(scope="session")
def grid2():
    from paper_2009_06635_b200 import workloads as W
    return W.grid_nnpdf_shaped()


@pytest.fixture(scope="session")
def ograph1(grid1):
    import oracle
    return oracle.OraclePdfGrid.from_spec(grid1)


@pytest.fixture(scope="session")
def ograph2(grid2):
    import oracle
    return oracle.OraclePdfGrid.from_spec(grid2)
