"""The parity criterion itself (tests/parity_util.py), on the CPU: the rule, the conditioning
clause with a full scale array and with a per-violator scale callable, chunked populations."""
import numpy as np
import pytest

import oracle
from paper_2009_06635_b200 import workloads as W
from parity_util import check_parity, check_parity_population, rule_violations


def test_rule_and_clause(grid2, ograph2, tmp_path, monkeypatch):
    monkeypatch.setenv("PDFB_PARITY_LOG", str(tmp_path / "log.jsonl"))
    pids = [21, 1, -3]
    x, q2 = W.queries_extrapolation_mix(grid2, 4001)
    ref, sc = ograph2.xfxq2(pids, x, q2, with_scale=True)
    assert check_parity(ref.copy(), ref)["n_clause"] == 0
    got = ref * (1 + 5e-13)                       # inside the rule wherever |ref| >= 1e-3 ...
    small = np.abs(ref) < 1e-3
    got[small] = ref[small] + 5e-16               # ... and where it is small
    assert not rule_violations(got, ref).any()
    got = ref.copy()
    got[1, 7] = ref[1, 7] * (1 + 3e-12) + 3e-15   # breaks the rule
    with pytest.raises(AssertionError):
        check_parity(got, ref)
    # ... and passes on the clause only if the scale allows it
    big = np.full_like(ref, 1e6)
    full = check_parity(got, ref, big, max_clause_frac=1.0)
    lazy = check_parity(got, ref, lambda cols: big[:, cols], max_clause_frac=1.0)
    assert full["n_clause"] == lazy["n_clause"] == 1 and full["max_d_over_S"] == lazy["max_d_over_S"] > 0
    with pytest.raises(AssertionError):
        check_parity(got, ref, np.full_like(ref, 1e-6), max_clause_frac=1.0)
    with pytest.raises(AssertionError):
        check_parity(got, ref, big, max_clause_frac=1e-9)
    # NaN patterns must agree
    got = ref.copy(); got[0, 3] = np.nan
    with pytest.raises(AssertionError):
        check_parity(got, ref)
    # chunked population = one call
    tot = check_parity_population(lambda a, b: ref[:, a:b], ograph2, pids, x, q2, chunk=1500, what="pop")
    assert tot["n"] == int((~np.isnan(ref)).sum()) and tot["n_clause"] == 0
    lines = (tmp_path / "log.jsonl").read_text().strip().splitlines()
    assert len(lines) >= 4 and '"what": "pop"' in lines[-1]


def test_slack_is_added_to_the_rule_only_where_given():
    """check_parity(slack=...): an output beyond the 1e-12 / 1e-15 rule passes iff the caller's derived
    allowance covers the excess; outputs with zero slack stay under the plain rule; uses are counted."""
    ref = np.array([[1.0, 2.0, 1e-6, 3.0]])
    got = ref + np.array([[5e-12, 0.0, 4e-15, 1e-13]])
    with pytest.raises(AssertionError):
        check_parity(got, ref, what="no slack", log=False)
    st = check_parity(got, ref, what="slack", log=False, slack=np.array([[5e-12, 0.0, 4e-15, 0.0]]))
    assert st["n_slack"] == 2 and st["n_clause"] == 0 and 0.7 < st["max_slack_used"] < 1.3   # (|d| / slack; the rule itself comes on top)
    with pytest.raises(AssertionError):   # the slack sits on the wrong outputs
        check_parity(got, ref, what="misplaced", log=False, slack=np.array([[0.0, 5e-12, 0.0, 4e-15]]))
