"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (one
pdf_xfxq2 call over the whole batch).  Configs 2, 4 and 5: EVERY output against the oracle
("parity is checked on all points"), the oracle run in chunks and its scale helper
only where the 1e-12 / 1e-15 rule breaks; the totals (max eq. 1 difference, rule
violations, clause uses) go to the parity log.  Config 3 (1e8 points x 11 flavours) too: all 1.1e9
outputs (`bench.py --parity` does the same check and puts the totals into the bench line)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2009_06635_b200 import binding as B, build, workloads as W
from parity_util import check_parity, check_parity_population


@pytest.fixture(scope="module")
def env(grid2):
    import torch
    assert torch.cuda.is_available()
    build.build()
    h = B.load_pdf_spec(grid2)
    assert B.pdf_grid_uses_smem_path(h)
    yield torch, h, oracle.OraclePdfGrid.from_spec(grid2)
    B.pdf_grid_free(h)


def _run(torch, h, pids, x, q2):
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    out = torch.full((len(pids), len(x)), float("nan"), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, pids, dx, dq, out)
    torch.cuda.synchronize()
    return out


def _population(torch, out, og, pids, x, q2, what, frac):
    st = check_parity_population(lambda a, b: out[:, a:b].cpu().numpy(), og, pids, x, q2,
                                 chunk=2_000_000, max_clause_frac=frac, what=what)
    print(what, st)
    return st


def test_config2_all_1e6_points(env, grid2):
    torch, h, og = env
    x, q2 = W.queries_in_range(grid2, 1_000_000, 2)
    pids = list(W.PIDS_11)
    out = _run(torch, h, pids, x, q2)
    st = _population(torch, out, og, pids, x, q2, "config2 all points", 2e-3)
    assert st["n"] == 11_000_000 and B.pdf_grid_status(h) == 0


def test_config3_all_1e8_points(env, grid2):
    """The headline configuration in the launch bench.py times: ONE pdf_xfxq2 call on 1e8 points x 11
    flavours, then every one of the 1.1e9 outputs against the oracle in chunks of 1e7 points
    (about two minutes of oracle on 16 cores)."""
    torch, h, og = env
    n = 100_000_000
    x, q2 = W.queries_in_range(grid2, n, 3)
    pids = list(W.PIDS_11)
    out = _run(torch, h, pids, x, q2)
    assert not bool(torch.isnan(out).any())          # every output written, none NaN in range
    assert B.pdf_grid_status(h) == 0
    st = check_parity_population(lambda a, b: out[:, a:b].cpu().numpy(), og, pids, x, q2,
                                 chunk=10_000_000, max_clause_frac=2e-3, what="config3 all points")
    print("config3", st)
    assert st["n"] == 11 * n and st["n_clause"] == 0
    del out
    torch.cuda.empty_cache()


@pytest.mark.parametrize("pids", [[21], list(W.PIDS_11)])
def test_config4_all_1e7_points(env, grid2, pids):
    torch, h, og = env
    x, q2 = W.queries_extrapolation_mix(grid2, 10_000_000)
    out = _run(torch, h, pids, x, q2)
    assert not bool(torch.isnan(out).any())
    st = _population(torch, out, og, pids, x, q2, f"config4 all points F={len(pids)}", 5e-3)
    assert st["n"] == 10_000_000 * len(pids)


def test_config5_all_1e7_events(env, grid2):
    torch, h, og = env
    x1, x2, q2 = W.queries_mc_events(grid2, 10_000_000)
    pids = list(W.PIDS_11)
    for name, x in (("x1", x1), ("x2", x2)):
        out = _run(torch, h, pids, x, q2)
        assert not bool(torch.isnan(out).any())
        _population(torch, out, og, pids, x, q2, f"config5 all events, {name}", 2e-3)
        del out
    aspec = W.make_alphas_grid()
    ha = B.load_alphas_spec(aspec)
    dq = torch.from_numpy(q2).cuda()
    a = torch.empty_like(dq)
    B.alphas_q2(ha, dq, a)
    torch.cuda.synchronize()
    st = check_parity(a.cpu().numpy(), oracle.OracleAlphas.from_spec(aspec).q2(q2), what="config5 alphas, all events")
    assert st["n"] == 10_000_000 and st["n_clause"] == 0
    B.alphas_grid_free(ha)
