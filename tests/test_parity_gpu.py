"""GPU parity: libpdfb200 (through the C-ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Sizes span many CTAs and a ragged tail; the oracle finishes each in
seconds."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2009_06635_b200 import binding as B, build, workloads as W
from parity_util import check_parity


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    build.build()
    B.lib()
    return torch


def gpu_xfxq2(torch, h, pids, x, q2):
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    out = torch.empty((len(pids), len(x)), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, pids, dx, dq, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.fixture(scope="module")
def h1(torch_cuda, grid1):
    h = B.load_pdf_spec(grid1)
    yield h
    B.pdf_grid_free(h)


@pytest.fixture(scope="module")
def h2(torch_cuda, grid2):
    h = B.load_pdf_spec(grid2)
    yield h
    B.pdf_grid_free(h)


def test_coordinate_ln_is_almost_always_correctly_rounded(torch_cuda):
    rng = np.random.default_rng(17)
    a = np.concatenate([np.exp(rng.uniform(np.log(1e-12), np.log(1e12), 400_000)),
                        1.0 + rng.uniform(-0.3, 0.4, 100_000), [1.0, 2.0, 0.5, 1e-300, 1e300, 5e-324]])
    d = torch_cuda.from_numpy(a).cuda()
    out = torch_cuda.empty_like(d)
    B.debug_ln(d, out)
    got = out.cpu().numpy()
    ref = np.array([oracle.ln(float(v)) for v in a])
    ulp = np.abs(got - ref) / np.spacing(np.abs(ref) + 1e-300)
    assert ulp.max() <= 1.0, ulp.max()
    frac = float((got != ref).mean())
    print("ln: fraction not correctly rounded", frac)
    assert frac < 0.02


def test_smem_path_is_the_one_that_runs(h1, h2):
    assert B.pdf_grid_uses_smem_path(h1) and B.pdf_grid_uses_smem_path(h2)


def test_knots_reproduced_exactly(torch_cuda, grid2, h2):
    for s in range(grid2.n_sub):
        q2 = grid2.sub_q(s) ** 2
        if s + 1 < grid2.n_sub:
            q2 = q2[:-1]
        X, Q = np.meshgrid(grid2.x_knots, q2, indexing="ij")
        got = gpu_xfxq2(torch_cuda, h2, grid2.pids, X.ravel().copy(), Q.ravel().copy())
        ref = grid2.sub_values(s)[:, : len(q2), :].transpose(2, 0, 1).reshape(grid2.n_pid, -1)
        assert np.array_equal(got, ref)


def test_config1_full(torch_cuda, grid1, ograph1, h1):
    x, q2 = W.queries_in_range(grid1, 10_000, 1)
    ref, sc = ograph1.xfxq2(grid1.pids, x, q2, with_scale=True)
    st = check_parity(gpu_xfxq2(torch_cuda, h1, grid1.pids, x, q2), ref, sc, what="config1")
    print("config1", st)


def test_config2_sample(torch_cuda, grid2, ograph2, h2):
    n = 300_007  # ragged tail
    x, q2 = W.queries_in_range(grid2, n, 2)
    ref, sc = ograph2.xfxq2(grid2.pids, x, q2, with_scale=True)
    st = check_parity(gpu_xfxq2(torch_cuda, h2, grid2.pids, x, q2), ref, sc, what="config2")
    print("config2", st)


def test_scan_crosses_every_knot_and_threshold(torch_cuda, grid2, ograph2, h2):
    x, q2 = W.scan_points(grid2, per_cell=2)
    pids = [21, -1, 2]
    ref, sc = ograph2.xfxq2(pids, x, q2, with_scale=True)
    st = check_parity(gpu_xfxq2(torch_cuda, h2, pids, x, q2), ref, sc, what="scan")
    print("scan", st)


@pytest.mark.parametrize("pids", [[21], list(W.PIDS_11)])
def test_config4_extrapolation_mix(torch_cuda, grid2, ograph2, h2, pids):
    n = 200_003
    x, q2 = W.queries_extrapolation_mix(grid2, n)
    ref, sc = ograph2.xfxq2(pids, x, q2, with_scale=True)
    st = check_parity(gpu_xfxq2(torch_cuda, h2, pids, x, q2), ref, sc, max_clause_frac=5e-3, what="config4")
    print("config4", len(pids), st)


def test_config5_events_and_alphas(torch_cuda, grid2, ograph2, h2):
    n = 150_001
    x1, x2, q2 = W.queries_mc_events(grid2, n)
    assert (q2 == grid2.q2_min).mean() > 0.15  # clipped events sit exactly on q_min (reading Q3)
    for x in (x1, x2):
        ref, sc = ograph2.xfxq2(grid2.pids, x, q2, with_scale=True)
        check_parity(gpu_xfxq2(torch_cuda, h2, grid2.pids, x, q2), ref, sc, what="config5")
    aspec = W.make_alphas_grid()
    oa = oracle.OracleAlphas.from_spec(aspec)
    ha = B.load_alphas_spec(aspec)
    dq = torch_cuda.from_numpy(q2).cuda()
    out = torch_cuda.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    torch_cuda.cuda.synchronize()
    check_parity(out.cpu().numpy(), oa.q2(q2), what="alphas config5")
    B.alphas_grid_free(ha)


def test_alphas_edges_thresholds_and_outside(torch_cuda):
    aspec = W.make_alphas_grid(jump=(1.0, 1.02, 1.0404, 1.061208))
    oa = oracle.OracleAlphas.from_spec(aspec)
    ha = B.load_alphas_spec(aspec)
    k2 = aspec.q_knots ** 2
    rng = np.random.default_rng(5)
    q2 = np.concatenate([k2, np.nextafter(k2, 0), np.nextafter(k2, np.inf),
                         np.exp(rng.uniform(np.log(0.1), np.log(1e12), 100_003)), [0.0, -1.0, np.nan]])
    dq = torch_cuda.from_numpy(q2).cuda()
    out = torch_cuda.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    torch_cuda.cuda.synchronize()
    check_parity(out.cpu().numpy(), oa.q2(q2), what="alphas edges")
    B.alphas_grid_free(ha)


def test_invalid_points_nan_and_counted(torch_cuda, grid1):
    h = B.load_pdf_spec(grid1)
    x = np.array([0.5, 1.0000001, 0.0, -0.1, np.nan, 0.5, 0.5, 0.5, np.inf, 0.5])
    q2 = np.array([10.0, 10.0, 10.0, 10.0, 10.0, 0.0, -3.0, np.nan, 10.0, np.inf])
    got = gpu_xfxq2(torch_cuda, h, grid1.pids, x, q2)
    og = oracle.OraclePdfGrid.from_spec(grid1)
    ref = og.xfxq2(grid1.pids, x, q2)
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    assert np.all(np.isnan(got[:, 1:])) and np.all(np.isfinite(got[:, 0]))
    assert B.pdf_grid_status(h) == og.n_invalid == 9
    B.pdf_grid_free(h)


def test_pid_alias_order_and_unknown(torch_cuda, grid1, h1):
    x, q2 = W.queries_in_range(grid1, 1000, 1)
    a = gpu_xfxq2(torch_cuda, h1, [0, 2, 1], x, q2)
    b = gpu_xfxq2(torch_cuda, h1, [1, 2, 21], x, q2)
    assert np.array_equal(a[0], b[2]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[0])
    with pytest.raises(B.PdfbError) as e:
        gpu_xfxq2(torch_cuda, h1, [6], x, q2)
    assert e.value.code == -3


def test_empty_batch_and_host_entry(torch_cuda, grid2, ograph2, h2):
    e = torch_cuda.empty(0, dtype=torch_cuda.float64, device="cuda")
    B.pdf_xfxq2(h2, [21], e, e, e)
    n = 5_000_011  # more than one pipeline chunk, ragged
    x, q2 = W.queries_in_range(grid2, n, 3)
    out = np.empty((2, n))
    B.pdf_xfxq2_host(h2, [21, 1], x, q2, out)
    dev = gpu_xfxq2(torch_cuda, h2, [21, 1], x, q2)
    assert np.array_equal(out, dev)
    idx = np.random.default_rng(1).choice(n, 50_000, replace=False)
    ref, sc = ograph2.xfxq2([21, 1], x[idx], q2[idx], with_scale=True)
    check_parity(out[:, idx], ref, sc, what="host entry")


def test_tiny_subgrids_two_and_three_knots(torch_cuda):
    from test_oracle_pins import make_spec, rand_knots
    rng = np.random.default_rng(2)
    xk = rand_knots(rng, 1e-4, 1.0, 3)
    subs = [rand_knots(rng, 1.5, 3.0, 2), rand_knots(rng, 3.0, 9.0, 3), rand_knots(rng, 9.0, 200.0, 4)]
    values = [rng.normal(size=(len(xk), len(q), 2)) for q in subs]
    spec = make_spec(xk, subs, [1, 21], values=values)
    og = oracle.OraclePdfGrid.from_spec(spec)
    h = B.load_pdf_spec(spec)
    x, q2 = W.scan_points(spec, per_cell=5)
    ref, sc = og.xfxq2([1, 21], x, q2, with_scale=True)
    check_parity(gpu_xfxq2(torch_cuda, h, [1, 21], x, q2), ref, sc, max_clause_frac=1.0, what="tiny")
    B.pdf_grid_free(h)
