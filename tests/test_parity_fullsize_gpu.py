"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (one
pdf_xfxq2 call over the whole batch): sampled outputs against the oracle, plus properties that
hold at any size (no NaN in range, every output written, invalid counter zero)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2009_06635_b200 import binding as B, build, workloads as W
from parity_util import check_parity


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


def _sample_check(torch, out, og, pids, x, q2, m, what, frac=2e-3):
    n = len(x)
    idx = np.unique(np.concatenate([np.random.default_rng(99).integers(0, n, m),
                                    np.arange(0, 4096), np.arange(n - 4096, n)]))
    got = out[:, torch.from_numpy(idx).cuda()].cpu().numpy()
    ref, sc = og.xfxq2(pids, x[idx], q2[idx], with_scale=True)
    st = check_parity(got, ref, sc, max_clause_frac=frac, what=what)
    print(what, st)
    return st


def test_config3_1e8_points_11_flavours(env, grid2):
    torch, h, og = env
    n = 100_000_000
    x, q2 = W.queries_in_range(grid2, n, 3)
    pids = list(W.PIDS_11)
    out = _run(torch, h, pids, x, q2)
    assert not bool(torch.isnan(out).any())          # every output written, none NaN in range
    assert B.pdf_grid_status(h) == 0
    _sample_check(torch, out, og, pids, x, q2, 300_000, "config3 full size")
    del out
    torch.cuda.empty_cache()


@pytest.mark.parametrize("pids", [[21], list(W.PIDS_11)])
def test_config4_1e7_points(env, grid2, pids):
    torch, h, og = env
    x, q2 = W.queries_extrapolation_mix(grid2, 10_000_000)
    out = _run(torch, h, pids, x, q2)
    assert not bool(torch.isnan(out).any())
    _sample_check(torch, out, og, pids, x, q2, 200_000, f"config4 full size F={len(pids)}", frac=5e-3)


def test_config5_1e7_events(env, grid2):
    torch, h, og = env
    x1, x2, q2 = W.queries_mc_events(grid2, 10_000_000)
    pids = list(W.PIDS_11)
    for x in (x1, x2):
        out = _run(torch, h, pids, x, q2)
        assert not bool(torch.isnan(out).any())
        _sample_check(torch, out, og, pids, x, q2, 100_000, "config5 full size")
    aspec = W.make_alphas_grid()
    ha = B.load_alphas_spec(aspec)
    dq = torch.from_numpy(q2).cuda()
    a = torch.empty_like(dq)
    B.alphas_q2(ha, dq, a)
    torch.cuda.synchronize()
    idx = np.random.default_rng(5).integers(0, len(q2), 200_000)
    check_parity(a[torch.from_numpy(idx).cuda()].cpu().numpy(), oracle.OracleAlphas.from_spec(aspec).q2(q2[idx]),
                 what="config5 alphas full size")
    B.alphas_grid_free(ha)
