"""GPU parity of the paths the main parity file does not reach ("parity coverage
holes"): the general alpha_s kernel (> 192 nodes), alphas_q2_host, the read-only-cache kernel
k_xfxq2_v0 forced on the NNPDF-shaped grid, and rule C's small-|y0| branch."""
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


def _alphas_points(aspec, rng, n):
    k2 = aspec.q_knots ** 2
    return np.concatenate([k2, np.nextafter(k2, 0), np.nextafter(k2, np.inf),
                           np.exp(rng.uniform(np.log(0.1), np.log(1e12), n)), [0.0, -1.0, np.nan, np.inf]])


def test_alphas_general_kernel_300_nodes(torch_cuda):
    """A 300-node list (> 192: k_alphas, binary search + weights4, not the replicated-line fast
    path), with discontinuities at the thresholds; nodes, their neighbours, outside, invalid."""
    torch = torch_cuda
    aspec = W.make_alphas_grid(nq_per_sub=(20, 40, 100, 140), jump=(1.0, 1.02, 1.0404, 1.061208))
    assert len(aspec.q_knots) == 300
    ha = B.load_alphas_spec(aspec)
    q2 = _alphas_points(aspec, np.random.default_rng(6), 200_003)
    dq = torch.from_numpy(q2).cuda()
    out, out_q = torch.empty_like(dq), torch.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    q = np.sqrt(np.where(q2 > 0, q2, np.nan))
    B.alphas_q(ha, torch.from_numpy(q).cuda(), out_q)
    torch.cuda.synchronize()
    oa = oracle.OracleAlphas.from_spec(aspec)
    st = check_parity(out.cpu().numpy(), oa.q2(q2), what="alphas 300 nodes (k_alphas)")
    assert st["n_clause"] == 0
    check_parity(out_q.cpu().numpy(), oa.q2(q * q), what="alphas_q 300 nodes (k_alphas)")
    B.alphas_grid_free(ha)
    # the largest list the library takes, and one node too many
    big = W.make_alphas_grid(nq_per_sub=(32, 64, 160, 256))
    hb = B.load_alphas_spec(big)
    q2 = _alphas_points(big, np.random.default_rng(7), 50_001)
    dq = torch.from_numpy(q2).cuda()
    out = torch.empty_like(dq)
    B.alphas_q2(hb, dq, out)
    torch.cuda.synchronize()
    check_parity(out.cpu().numpy(), oracle.OracleAlphas.from_spec(big).q2(q2), what="alphas 512 nodes")
    B.alphas_grid_free(hb)
    with pytest.raises(B.PdfbError):
        B.load_alphas_spec(W.make_alphas_grid(nq_per_sub=(32, 64, 160, 257)))


def test_alphas_fast_path_dense_nodes(torch_cuda):
    """The replicated-line fast path (<= 192 nodes) with its table-based logarithm on a dense list:
    190 nodes, i.e. ln Q^2 spacings down to 0.02 (the tolerance budget of that logarithm scales with
    the spacing, pdfb_internal.cuh); nodes, their neighbours, thresholds with jumps, outside."""
    torch = torch_cuda
    aspec = W.make_alphas_grid(nq_per_sub=(40, 50, 50, 50), jump=(1.0, 0.97, 1.01, 1.03))
    assert len(aspec.q_knots) == 190
    assert np.diff(np.log(aspec.q_knots[:40] ** 2)).min() < 0.025
    ha = B.load_alphas_spec(aspec)
    q2 = _alphas_points(aspec, np.random.default_rng(9), 400_003)
    dq = torch.from_numpy(q2).cuda()
    out = torch.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    torch.cuda.synchronize()
    st = check_parity(out.cpu().numpy(), oracle.OracleAlphas.from_spec(aspec).q2(q2), what="alphas 190 nodes (fast path)")
    assert st["n_clause"] == 0 and st["max_eq1"] < 2e-13
    B.alphas_grid_free(ha)


@pytest.mark.parametrize("nodes", [(6, 12, 30, 52), (20, 40, 100, 140)])
def test_alphas_q2_host_entry(torch_cuda, nodes):
    """alphas_q2_host (host buffers, chunked pipeline): bit-identical to alphas_q2 on the same
    points, more than one pipeline chunk with a ragged tail, and within tolerance of the oracle."""
    torch = torch_cuda
    aspec = W.make_alphas_grid(nq_per_sub=nodes)
    ha = B.load_alphas_spec(aspec)
    n = 9_000_011
    rng = np.random.default_rng(8)
    q2 = np.exp(rng.uniform(np.log(0.5), np.log(4e10), n))
    q2[:5] = [0.0, -1.0, np.nan, aspec.q_knots[0] ** 2, aspec.q_knots[-1] ** 2]
    out_h = np.empty(n)
    B.alphas_q2_host(ha, q2, out_h)
    dq = torch.from_numpy(q2).cuda()
    out_d = torch.empty_like(dq)
    B.alphas_q2(ha, dq, out_d)
    torch.cuda.synchronize()
    assert np.array_equal(out_h, out_d.cpu().numpy(), equal_nan=True)
    idx = np.concatenate([np.arange(64), rng.integers(0, n, 200_000), np.arange(n - 64, n)])
    check_parity(out_h[idx], oracle.OracleAlphas.from_spec(aspec).q2(q2[idx]), what=f"alphas_q2_host {sum(nodes)} nodes")
    B.alphas_q2_host(ha, q2[:0], out_h[:0])      # empty batch
    B.alphas_grid_free(ha)


def test_forced_fallback_kernel_on_the_nnpdf_grid(torch_cuda, grid2, ograph2, monkeypatch):
    """PDFB_FORCE_FALLBACK=1 at load: k_xfxq2_v0 (one thread per point, read-only cache) on the
    NNPDF-shaped grid -- the config-4 mix, the knot/threshold scan, PID subsets, the Q entry."""
    torch = torch_cuda
    monkeypatch.setenv("PDFB_FORCE_FALLBACK", "1")
    h = B.load_pdf_spec(grid2)
    monkeypatch.delenv("PDFB_FORCE_FALLBACK")
    assert not B.pdf_grid_uses_smem_path(h)
    pids = list(W.PIDS_11)
    x, q2 = W.queries_extrapolation_mix(grid2, 150_007)
    xs, qs = W.scan_points(grid2, per_cell=2)
    x, q2 = np.concatenate([x, xs]), np.concatenate([q2, qs])
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    for req in (pids, [21], [0, -5, 3, 3]):
        out = torch.empty((len(req), len(x)), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h, req, dx, dq, out)
        torch.cuda.synchronize()
        ref, sc = ograph2.xfxq2(req, x, q2, with_scale=True)
        st = check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"forced k_xfxq2_v0 {req}")
        print("fallback", req, st)
    out_q = torch.empty((len(pids), len(x)), dtype=torch.float64, device="cuda")
    out_2 = torch.empty_like(out_q)
    q = np.sqrt(q2)
    B.pdf_xfxq(h, pids, dx, torch.from_numpy(q).cuda(), out_q)
    B.pdf_xfxq2(h, pids, dx, torch.from_numpy(q * q).cuda(), out_2)
    torch.cuda.synchronize()
    assert torch.equal(out_q, out_2)
    # knots reproduced bit for bit on this path too
    X, Q = np.meshgrid(grid2.x_knots, grid2.sub_q(1) ** 2, indexing="ij")
    out = torch.empty((len(pids), X.size), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, pids, torch.from_numpy(X.ravel().copy()).cuda(), torch.from_numpy(Q.ravel().copy()).cuda(), out)
    assert np.array_equal(out.cpu().numpy(), grid2.sub_values(1).transpose(2, 0, 1).reshape(len(pids), -1))
    B.pdf_grid_free(h)


@pytest.mark.parametrize("force_fallback", [False, True])
def test_rule_C_small_y0_branch(torch_cuda, monkeypatch, force_fallback):
    """Q^2 < q_min with |y0| on either side of 1e-5 (reading Q9: gamma = 1 below it): a grid whose
    q_min row crosses 1e-5 along x, so both branches occur in one batch, on both kernels."""
    torch = torch_cuda
    from test_oracle_pins import make_spec
    xk = np.geomspace(1e-5, 1.0, 24)
    qk = np.geomspace(1.5, 300.0, 9)

    def fn(s, x, q2, pid):
        amp = 3e-4 if pid == 21 else -2e-4
        return amp * x ** 0.4 * (1.0 - x) ** 2 * (q2 / qk[0] ** 2) ** (0.25 if pid == 21 else -0.6)

    spec = make_spec(xk, [qk], [1, 21], fn)
    if force_fallback:
        monkeypatch.setenv("PDFB_FORCE_FALLBACK", "1")
    h = B.load_pdf_spec(spec)
    monkeypatch.delenv("PDFB_FORCE_FALLBACK", raising=False)
    assert bool(B.pdf_grid_uses_smem_path(h)) != force_fallback
    rng = np.random.default_rng(3)
    n = 60_001
    x = np.exp(rng.uniform(np.log(1e-7), 0.0, n))
    q2 = spec.q2_min * np.exp(rng.uniform(np.log(1e-3), 0.0, n)) * (1 - 1e-12)
    og = oracle.OraclePdfGrid.from_spec(spec)
    y0 = og.xfxq2([1, 21], np.clip(x, xk[0], 1.0), np.full(n, spec.q2_min))
    frac_small = (np.abs(y0) < 1e-5).mean()
    assert 0.2 < frac_small < 0.8, frac_small       # both branches are well populated
    out = torch.empty((2, n), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, [1, 21], torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), out)
    torch.cuda.synchronize()
    ref, sc = og.xfxq2([1, 21], x, q2, with_scale=True)
    st = check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"rule C small y0, fallback={force_fallback}")
    print(st)
    B.pdf_grid_free(h)


@pytest.mark.parametrize("force_fallback", [False, True])
def test_point_major_and_fp32_output(torch_cuda, grid2, ograph2, monkeypatch, force_fallback):
    """pdf_xfxq2_pm / pdf_xfxq2_f32: compile-time variants of the same
    kernels.  Point-major: bit-identical to pdf_xfxq2 transposed.  fp32: the fp64 result of pdf_xfxq2
    rounded once (bit-identical to casting it), hence within half an fp32 ulp + the fp64 tolerance of
    the oracle.  The extrapolation mix (class lists), the scan, PID subsets over 1-3 groups and the
    2-column plan; both kernels."""
    torch = torch_cuda
    if force_fallback:
        monkeypatch.setenv("PDFB_FORCE_FALLBACK", "1")
    h = B.load_pdf_spec(grid2)
    monkeypatch.delenv("PDFB_FORCE_FALLBACK", raising=False)
    assert bool(B.pdf_grid_uses_smem_path(h)) != force_fallback
    x, q2 = W.queries_extrapolation_mix(grid2, 120_011)
    xs, qs = W.scan_points(grid2, per_cell=1)
    x, q2 = np.concatenate([x, xs, [0.5, -1.0, 2.0]]), np.concatenate([q2, qs, [np.nan, 10.0, 10.0]])
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    n = len(x)
    for req in (list(W.PIDS_11), [21], [3, -5, 0, 3, 1]):
        fm = torch.empty((len(req), n), dtype=torch.float64, device="cuda")
        pm = torch.full((n, len(req)), 7.0, dtype=torch.float64, device="cuda")
        f32 = torch.full((len(req), n), 7.0, dtype=torch.float32, device="cuda")
        B.pdf_xfxq2(h, req, dx, dq, fm)
        B.pdf_xfxq2_pm(h, req, dx, dq, pm)
        B.pdf_xfxq2_f32(h, req, dx, dq, f32)
        torch.cuda.synchronize()
        assert torch.equal(torch.nan_to_num(pm.t().contiguous(), nan=-9.0), torch.nan_to_num(fm, nan=-9.0))
        assert torch.equal(torch.nan_to_num(f32, nan=-9.0), torch.nan_to_num(fm.to(torch.float32), nan=-9.0))
        ref, sc = ograph2.xfxq2(req, x, q2, with_scale=True)
        check_parity(pm.t().cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"point-major {req} fallback={force_fallback}")
        got32 = f32.cpu().numpy().astype(np.float64)
        ok = ~np.isnan(ref)
        assert np.array_equal(np.isnan(got32), np.isnan(ref))
        half_ulp32 = 0.5 * np.spacing(np.abs(ref[ok]).astype(np.float32)).astype(np.float64)
        assert np.all(np.abs(got32[ok] - ref[ok]) <= half_ulp32 + 1e-12 * np.abs(ref[ok]) + 1e-15 + 1e-12 * sc[ok])
    B.pdf_grid_free(h)


def test_per_subgrid_x_knot_arrays(torch_cuda, tmp_path):
    """pdf_grid_load_xs ("allowing per-subgrid x-knot arrays"): sub-grids
    with 100 / 80 / 34 / 120 x knots on one Q^2 layout, loaded directly and from a member file in the
    LHAPDF text layout; every knot of every sub-grid exactly, random points in and outside the grid,
    pdf_lumi_events, the Q entry point and the output variants; identical arrays give an ordinary handle."""
    torch = torch_cuda
    base = W.grid_nnpdf_shaped()
    xs = [base.x_knots, W._geomspace(1e-9, 1.0, 80), base.x_knots[::3].copy(), W._geomspace(1e-9, 1.0, 120)]
    spec = W.make_pdf_grid_xs(xs, (1.65, (1.65 * 4.92) ** 0.5, 4.92, 172.5, 1.0e5), (7, 14, 23, 20), W.PIDS_11)
    og = oracle.OraclePdfGrid.from_spec(spec)
    h = B.load_pdf_spec(spec)
    assert not B.pdf_grid_uses_smem_path(h)
    pids = list(W.PIDS_11)

    def run(x, q2, req=pids):
        out = torch.empty((len(req), len(x)), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h, req, torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), out)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    for s in range(spec.n_sub):   # knots reproduced bit for bit; a threshold belongs to the upper sub-grid
        q = spec.sub_q(s) if s + 1 == spec.n_sub else spec.sub_q(s)[:-1]
        X, Q = np.meshgrid(spec.sub_x(s), q ** 2, indexing="ij")
        ref = spec.sub_values(s)[:, :len(q), :].transpose(2, 0, 1).reshape(len(pids), -1)
        got = run(X.ravel().copy(), Q.ravel().copy())
        assert np.array_equal(got, ref)   # x_max and q2_max included: t = 1 exactly on the last knot
    x, q2 = W.queries_extrapolation_mix(base, 150_011)
    ref, sc = og.xfxq2(pids, x, q2, with_scale=True)
    st = check_parity(run(x, q2), ref, sc, max_clause_frac=5e-3, what="per-sub-grid x knots, mix")
    print(st)
    sub = [21, -3, 0]
    rs, ss = og.xfxq2(sub, x, q2, with_scale=True)
    check_parity(run(x, q2, sub), rs, ss, max_clause_frac=5e-3, what="per-sub-grid x knots, PID subset")
    # the fused call goes through the general kernel on such a grid
    n = 40_001
    x1, x2, qe = W.queries_mc_events(base, n)
    terms = [(1, -1, 1.0), (-2, 2, 0.5), (21, 21, 0.25), (21, 3, -1.0)]
    lum = torch.empty(n, dtype=torch.float64, device="cuda")
    B.pdf_lumi_events(h, terms, torch.from_numpy(x1).cuda(), torch.from_numpy(x2).cuda(), torch.from_numpy(qe).cuda(), lum)
    torch.cuda.synchronize()
    lr, ls = oracle.lumi_events(og, terms, x1, x2, qe, with_scale=True)
    check_parity(lum.cpu().numpy(), lr, ls, what="per-sub-grid x knots, lumi")
    # the same member through a file in the LHAPDF text layout
    d = tmp_path / "xsset"
    d.mkdir()
    W.write_lhagrid(spec, str(d / "xsset_0000.dat"))
    W.write_lhapdf_info(str(d / "xsset.info"), 1, pids, W.make_alphas_grid())
    hf, ha, fp = B.load_lhapdf_set(str(d))
    o1 = torch.empty((len(pids), len(x)), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(hf, pids, torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), o1)
    torch.cuda.synchronize()
    assert np.array_equal(o1.cpu().numpy(), run(x, q2), equal_nan=True) and list(fp) == pids
    B.pdf_grid_free(hf); B.alphas_grid_free(ha); B.pdf_grid_free(h)
    # identical arrays passed per sub-grid: an ordinary (shared-memory) handle, same numbers as pdf_grid_load
    same = B.pdf_grid_load_xs(np.arange(5, dtype=np.int32) * base.nx, np.tile(base.x_knots, 4), base.q_offsets,
                              base.q_knots, base.pids, base.values)
    plain = B.load_pdf_spec(base)
    assert B.pdf_grid_uses_smem_path(same)
    a = torch.empty((len(pids), len(x)), dtype=torch.float64, device="cuda"); b = torch.empty_like(a)
    B.pdf_xfxq2(same, pids, torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), a)
    B.pdf_xfxq2(plain, pids, torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), b)
    torch.cuda.synchronize()
    assert torch.equal(torch.nan_to_num(a, nan=-9.0), torch.nan_to_num(b, nan=-9.0))
    B.pdf_grid_free(same); B.pdf_grid_free(plain)
    # arrays that do not span one common x range are refused
    bad = [base.x_knots, W._geomspace(1e-8, 1.0, 80), base.x_knots, base.x_knots]
    sb = W.make_pdf_grid_xs(bad, (1.65, (1.65 * 4.92) ** 0.5, 4.92, 172.5, 1.0e5), (7, 14, 23, 20), W.PIDS_11)
    with pytest.raises(B.PdfbError) as e:
        B.load_pdf_spec(sb)
    assert e.value.code == B.PDFB_EKNOTS
