"""GPU parity of pdf_lumi_events (events with x1, x2 and one
shared Q^2) against the oracle helper oracle.lumi_events (the single-point oracle twice + the sum).

Tolerance: the north_star rule on the luminosity itself; where it breaks, the
conditioning clause with the first-order scale of the bilinear form, S = sum_t |c_t| (S_a |xf_b| +
|xf_a| S_b): a sum of signed products cancels like a single interpolant does."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2009_06635_b200 import binding as B, build, workloads as W
from parity_util import check_parity

QQBAR_GG = [(q, -q, 1.0) for q in (1, 2, 3, 4, 5)] + [(-q, q, 1.0) for q in (1, 2, 3, 4, 5)] + [(21, 21, 0.25)]


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    build.build()
    B.lib()
    return torch


def gpu_lumi(torch, h, terms, x1, x2, q2, ha=None, divide=False):
    d1, d2, dq = (torch.from_numpy(a).cuda() for a in (x1, x2, q2))
    out = torch.full((len(x1),), 7.0, dtype=torch.float64, device="cuda")
    aout = torch.empty_like(out) if ha is not None else None
    B.pdf_lumi_events(h, terms, d1, d2, dq, out, alphas=ha, alphas_out=aout, divide_by_x=divide)
    torch.cuda.synchronize()
    return out.cpu().numpy(), (aout.cpu().numpy() if ha is not None else None)


def dense_terms(pids, rng):
    return [(a, b, float(c)) for a in pids for b in pids for c in [rng.normal()] if rng.uniform() < 0.7]


def check_lumi(got, og, terms, x1, x2, q2, what, divide=False, frac=2e-3):
    ref, sc = oracle.lumi_events(og, terms, x1, x2, q2, divide_by_x=divide, with_scale=True)
    st = check_parity(got, ref, sc, max_clause_frac=frac, what=what)
    print(what, st)
    return st


def test_config5_events(torch_cuda, grid2, ograph2):
    """Config 5's events (a quarter sit exactly on q_min), three pair tables, both output forms, alpha_s
    in the same call; band kernel with 6 column pairs."""
    torch = torch_cuda
    h = B.load_pdf_spec(grid2)
    aspec = W.make_alphas_grid()
    ha = B.load_alphas_spec(aspec)
    n = 200_003
    x1, x2, q2 = W.queries_mc_events(grid2, n)
    rng = np.random.default_rng(12)
    for name, terms in (("qqbar+gg", QQBAR_GG), ("dense", dense_terms(W.PIDS_11, rng)), ("one term, PID 0", [(0, 2, -3.5)])):
        got, al = gpu_lumi(torch, h, terms, x1, x2, q2, ha=ha)
        check_lumi(got, ograph2, terms, x1, x2, q2, f"lumi config5 {name}")
        check_parity(al, oracle.OracleAlphas.from_spec(aspec).q2(q2), what="lumi config5 alphas")
    got, _ = gpu_lumi(torch, h, QQBAR_GG, x1, x2, q2, divide=True)
    check_lumi(got, ograph2, QQBAR_GG, x1, x2, q2, "lumi config5 f f form", divide=True)
    # the same numbers as the unfused calls + the caller's contraction, to rounding
    pids = list(W.PIDS_11)
    f1 = torch.empty((11, n), dtype=torch.float64, device="cuda"); f2 = torch.empty_like(f1)
    B.pdf_xfxq2(h, pids, torch.from_numpy(x1).cuda(), torch.from_numpy(q2).cuda(), f1)
    B.pdf_xfxq2(h, pids, torch.from_numpy(x2).cuda(), torch.from_numpy(q2).cuda(), f2)
    acc = torch.zeros(n, dtype=torch.float64, device="cuda")
    for a, b, c in QQBAR_GG:
        acc += c * f1[pids.index(a)] * f2[pids.index(b)]
    got, _ = gpu_lumi(torch, h, QQBAR_GG, x1, x2, q2)
    ref, sc = oracle.lumi_events(ograph2, QQBAR_GG, x1, x2, q2, with_scale=True)
    assert np.all(np.abs(got - acc.cpu().numpy()) <= 1e-12 * sc)
    B.pdf_grid_free(h)
    B.alphas_grid_free(ha)


def test_scan_every_cell_and_band_edge(torch_cuda, grid2, ograph2):
    """Every Q^2 knot, threshold and interval (band boundaries included) against every x interval."""
    torch = torch_cuda
    h = B.load_pdf_spec(grid2)
    x, q2 = W.scan_points(grid2, per_cell=1)
    rng = np.random.default_rng(3)
    x2 = rng.permutation(x)
    terms = dense_terms(W.PIDS_11, rng)
    got, _ = gpu_lumi(torch, h, terms, x, x2, q2)
    check_lumi(got, ograph2, terms, x, x2, q2, "lumi scan")
    B.pdf_grid_free(h)


def test_events_outside_the_grid_and_invalid(torch_cuda, grid2, ograph2):
    """Events with a point outside the grid take the general kernel (continuation rules on either
    beam); coordinates without a value give NaN and are counted once per event; empty batch."""
    torch = torch_cuda
    h = B.load_pdf_spec(grid2)
    n = 60_001
    x1, q2 = W.queries_extrapolation_mix(grid2, n)
    x2 = np.random.default_rng(5).permutation(x1)
    terms = QQBAR_GG
    got, _ = gpu_lumi(torch, h, terms, x1, x2, q2)
    check_lumi(got, ograph2, terms, x1, x2, q2, "lumi extrapolation mix", frac=5e-3)
    before = B.pdf_grid_status(h)
    bx1 = np.array([0.1, 1.5, 0.1, 0.1, np.nan, 0.1]); bx2 = np.array([0.2, 0.2, -1.0, 0.2, 0.2, 0.2])
    bq = np.array([10.0, 10.0, 10.0, 0.0, 10.0, np.inf])
    got, _ = gpu_lumi(torch, h, terms, bx1, bx2, bq)
    assert np.isfinite(got[0]) and np.isnan(got[1:]).all()
    assert B.pdf_grid_status(h) - before == 5
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    B.pdf_lumi_events(h, terms, e, e, e, e)
    with pytest.raises(B.PdfbError) as err:
        B.pdf_lumi_events(h, [(6, 1, 1.0)], e, e, e, e)
    assert err.value.code == B.PDFB_EPID
    B.pdf_grid_free(h)


@pytest.mark.parametrize("which", ["config1 (3 PIDs)", "member grid (13 PIDs)", "fallback (general kernel)"])
def test_other_grids(torch_cuda, grid1, grid2, which, monkeypatch):
    """2 column pairs in one band (config 1), 7 pairs (13 PIDs), and a grid the shared-memory path does
    not take (every event through the general kernel)."""
    torch = torch_cuda
    rng = np.random.default_rng(8)
    if which.startswith("config1"):
        spec = grid1
    elif which.startswith("member"):
        spec = W.grid_member(1)
    else:
        spec = grid2
        monkeypatch.setenv("PDFB_FORCE_FALLBACK", "1")
    h = B.load_pdf_spec(spec)
    monkeypatch.delenv("PDFB_FORCE_FALLBACK", raising=False)
    og = oracle.OraclePdfGrid.from_spec(spec)
    n = 50_003
    x1 = np.exp(rng.uniform(np.log(spec.x_knots[0]), 0.0, n)); x2 = np.exp(rng.uniform(np.log(spec.x_knots[0]), 0.0, n))
    q2 = np.clip(np.exp(rng.uniform(np.log(spec.q2_min), np.log(spec.q2_max), n)), spec.q2_min, spec.q2_max)
    x1, x2 = np.clip(x1, spec.x_knots[0], 1.0), np.clip(x2, spec.x_knots[0], 1.0)
    terms = dense_terms([int(p) for p in spec.pids], rng)
    got, _ = gpu_lumi(torch, h, terms, x1, x2, q2)
    check_lumi(got, og, terms, x1, x2, q2, f"lumi {which}")
    B.pdf_grid_free(h)


def test_config5_all_1e7_events(torch_cuda, grid2, ograph2):
    """Full size, every event (the oracle in chunks, its scale only where the rule breaks)."""
    torch = torch_cuda
    h = B.load_pdf_spec(grid2)
    n = 10_000_000
    x1, x2, q2 = W.queries_mc_events(grid2, n)
    got, _ = gpu_lumi(torch, h, QQBAR_GG, x1, x2, q2)
    tot = {"n": 0, "n_clause": 0, "max_eq1": 0.0}
    for a in range(0, n, 2_000_000):
        s = slice(a, a + 2_000_000)
        ref = oracle.lumi_events(ograph2, QQBAR_GG, x1[s], x2[s], q2[s])
        xa, xb, qa = x1[s], x2[s], q2[s]
        st = check_parity(got[s], ref, lambda c: oracle.lumi_events(ograph2, QQBAR_GG, xa[c], xb[c], qa[c], with_scale=True)[1],
                          what="lumi config5 all events", log=(a == 0))
        tot["n"] += st["n"]; tot["n_clause"] += st["n_clause"]; tot["max_eq1"] = max(tot["max_eq1"], st["max_eq1"])
    print("lumi all events", tot)
    assert tot["n"] == n and tot["n_clause"] <= 2e-3 * n
    B.pdf_grid_free(h)
