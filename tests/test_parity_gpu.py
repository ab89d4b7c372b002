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


@pytest.mark.parametrize("n_nodes", [100, 240])  # table-logarithm kernel (<= 192 nodes) and the general one
def test_alphas_on_a_node_is_the_node_value(torch_cuda, n_nodes):
    """include/pdfb200.h: a query on a knot returns the table value bit for bit -- for alpha_s too, in
    both kernels, the LAST node included (at a flavour threshold, stored twice, the upper copy)."""
    per = n_nodes // 4
    aspec = W.make_alphas_grid(nq_per_sub=(per, per, per, n_nodes - 3 * per), jump=(1.0, 1.02, 1.0404, 1.061208))
    ha = B.load_alphas_spec(aspec)
    k2 = aspec.q_knots ** 2
    dq = torch_cuda.from_numpy(k2).cuda()
    out = torch_cuda.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    torch_cuda.cuda.synchronize()
    want = aspec.alphas.copy()
    rep = np.nonzero(k2[1:] == k2[:-1])[0]          # lower copy of a threshold: the query lands on the upper one
    want[rep] = aspec.alphas[rep + 1]
    assert np.array_equal(out.cpu().numpy(), want)
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
    check_parity(gpu_xfxq2(torch_cuda, h, [1, 21], x, q2), ref, sc, what="tiny")  # measured: no output needs the clause
    B.pdf_grid_free(h)


def graded_knots(rng, lo, hi, n_regular, cluster, at):
    """Knots on [lo, hi]: random ln-gaps with a cluster of small gaps spliced in at index `at`;
    neighbouring gaps differ by at most ~4x (as in real grids), so derivative coefficients stay O(1)."""
    gaps = list(rng.uniform(0.45, 1.0, n_regular))
    gaps[at:at] = list(cluster)
    gaps = np.asarray(gaps) * (np.log(hi / lo) / np.sum(gaps))
    k = lo * np.exp(np.concatenate([[0.0], np.cumsum(gaps)]))
    k[-1] = hi
    return k


def test_irregular_grid_on_the_smem_path(torch_cuda):
    """Non-uniform knots with dense clusters (several knots per search-LUT bin), nx not a multiple
    of 4, 4-knot sub-grids next to long ones, random values of both signs: every cell, knot and
    threshold is scanned, plus out-of-grid points, for PID subsets that use 1, 2 and 3 flavour
    groups, duplicates and PID 0.  The smallest gaps are 0.01 (ln Q^2) and 0.02 (ln x) against >= 0.09
    in the paper-shaped grids: one ulp of u (|u| <= 16: 3.6e-15) moves t by up to 3.6e-13, and the
    weights change by up to ~4 per unit t next to a 4x narrower neighbour, per axis, so the
    conditioning clause is taken at 4e-12 * S here; the plain rule is unchanged."""
    from test_oracle_pins import make_spec, rand_knots
    rng = np.random.default_rng(77)
    xk = graded_knots(rng, 1e-7, 1.0, 21, [0.25, 0.08, 0.025, 0.02, 0.02, 0.02, 0.025, 0.08, 0.25], 9)
    assert len(xk) == 31 and len(xk) % 4 != 0
    subs = [np.geomspace(1.3, 2.0, 4), graded_knots(rng, 2.0, 4.5, 8, [], 0), np.geomspace(4.5, 4.75, 4),
            graded_knots(rng, 4.75, 3e3, 10, [0.15, 0.05, 0.018, 0.006, 0.006, 0.006, 0.018, 0.05, 0.15], 4)]
    lutbin = np.log((3e3 / 1.3) ** 2) / 512
    assert (np.diff(2 * np.log(subs[3])) < lutbin / 2).sum() >= 3      # several knots share a LUT bin
    assert (np.diff(np.log(xk)) < np.log(1e7) / 512 / 1.2).sum() >= 3
    pids_all = [-3, -2, -1, 1, 2, 3, 4, 21, 22]
    values = [rng.normal(size=(len(xk), len(q), len(pids_all))) for q in subs]
    spec = make_spec(xk, subs, pids_all, values=values)
    og = oracle.OraclePdfGrid.from_spec(spec)
    h = B.load_pdf_spec(spec)
    assert B.lib().pdf_grid_uses_smem_path(h) == 1
    x, q2 = W.scan_points(spec, per_cell=3)
    lo, hi = float(subs[0][0]) ** 2, float(subs[-1][-1]) ** 2
    xo = np.exp(rng.uniform(np.log(1e-9), 0.0, 4000)); qo = np.exp(rng.uniform(np.log(lo / 4), np.log(hi * 4), 4000))
    x, q2 = np.concatenate([x, xo]), np.concatenate([q2, qo])
    for req in ([21], [0, 22], [4, -3, 1], pids_all, [2, 2, 21, -1, 3, 22, 2]):
        ref, sc = og.xfxq2(req, x, q2, with_scale=True)
        check_parity(gpu_xfxq2(torch_cuda, h, req, x, q2), ref, sc, max_clause_frac=4e-4, what=f"irregular {req}", clause_rel=4e-12)  # measured 1.2e-4 .. 1.5e-4 of the outputs (parity log)
    B.pdf_grid_free(h)


def test_q_argument_entry_points(torch_cuda, grid2, ograph2, h2):
    """pdf_xfxq / alphas_q (the second interpolating method of each quantity) are
    defined as the Q^2 methods at Q*Q rounded once: bit-identical to pdf_xfxq2 / alphas_q2 on the
    squared scales of the same batch, and within tolerance of the oracle at those scales; Q <= 0 and
    NaN give NaN and are counted."""
    torch = torch_cuda
    pids = list(W.PIDS_11)
    x, q2 = W.queries_extrapolation_mix(grid2, 60_001)
    q = np.sqrt(q2)
    qq = q * q
    dx, dq, dqq = (torch.from_numpy(a).cuda() for a in (x, q, qq))
    out_q = torch.empty((len(pids), len(x)), dtype=torch.float64, device="cuda")
    out_q2 = torch.empty_like(out_q)
    B.pdf_xfxq(h2, pids, dx, dq, out_q)
    B.pdf_xfxq2(h2, pids, dx, dqq, out_q2)
    torch.cuda.synchronize()
    a, b = out_q.cpu().numpy(), out_q2.cpu().numpy()
    assert np.array_equal(a, b, equal_nan=True)
    ref, sc = ograph2.xfxq2(pids, x, qq, with_scale=True)
    check_parity(a, ref, sc, max_clause_frac=5e-3, what="xfxq")
    # no value for Q <= 0, NaN
    before = B.pdf_grid_status(h2)
    bx = torch.tensor([0.1, 0.1, 0.1, 0.1], dtype=torch.float64, device="cuda")
    bq = torch.tensor([0.0, -2.0, float("nan"), 10.0], dtype=torch.float64, device="cuda")
    bo = torch.empty((len(pids), 4), dtype=torch.float64, device="cuda")
    B.pdf_xfxq(h2, pids, bx, bq, bo)
    bo = bo.cpu().numpy()
    assert np.isnan(bo[:, :3]).all() and np.isfinite(bo[:, 3]).all()
    assert B.pdf_grid_status(h2) - before == 3
    aspec = W.make_alphas_grid()
    ha = B.load_alphas_spec(aspec)
    ra, rb, rc = torch.empty_like(dq), torch.empty_like(dq), torch.empty_like(bq)
    B.alphas_q(ha, dq, ra)
    B.alphas_q2(ha, dqq, rb)
    B.alphas_q(ha, bq, rc)
    torch.cuda.synchronize()
    ra, rb, rc = ra.cpu().numpy(), rb.cpu().numpy(), rc.cpu().numpy()
    assert np.array_equal(ra, rb)
    assert np.isnan(rc[:3]).all() and np.isfinite(rc[3])
    check_parity(ra, oracle.OracleAlphas.from_spec(aspec).q2(qq), what="alphas_q")
    B.alphas_grid_free(ha)


def test_member_set(torch_cuda):
    """pdf_set_load / pdf_xfxq2_members (Table 2 shape: 13 flavours, 2415 x-points
    at the fitting scale, N_rep members): every member against the single-member oracle on its own
    table, member ranges, more jobs than SMs (one CTA per job) and fewer (persistent CTAs), the
    extrapolation mix, and pdf_xfxq2 = member 0."""
    torch = torch_cuda
    n_mem = 60                                   # 60 members x 4 flavour groups = 240 jobs > 148 SMs
    g0 = W.grid_member(0)
    vals = W.member_values(n_mem)
    h = B.pdf_set_load(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals)
    assert B.pdf_set_members(h) == n_mem and B.pdf_grid_uses_smem_path(h)
    pids = list(W.PIDS_13)
    x, q2 = W.queries_fk_xgrid(g0)
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    out = torch.empty((n_mem, len(pids), len(x)), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2_members(h, 0, n_mem, pids, dx, dq, out)
    torch.cuda.synchronize()
    ref, sc = oracle.xfxq2_members(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals, pids, x, q2, with_scale=True)
    check_parity(out.cpu().numpy(), ref, sc, what="member set, FK x-grid")
    # the set kernel keeps the points' (cell, t, tau) in shared memory across its jobs; a member loaded
    # on its own goes through the ordinary loop: same lanes, same arithmetic, so bit for bit the same
    for m in (0, 5, n_mem - 1):
        h1 = B.pdf_grid_load(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals[m])
        o1 = torch.empty((len(pids), len(x)), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h1, pids, dx, dq, o1)
        torch.cuda.synchronize()
        assert torch.equal(o1.view(torch.int64), out[m].view(torch.int64)), m
        B.pdf_grid_free(h1)
    # a batch with invalid points (no value: NaN, counted once per point) still takes the cached path
    xb, qb = x.copy(), q2.copy()
    xb[[3, 700, 2414]] = [np.nan, 1.5, -1.0]
    qb[[9, 1000]] = [0.0, np.inf]
    ob = torch.empty((n_mem, len(pids), len(x)), dtype=torch.float64, device="cuda")
    before = B.pdf_grid_status(h)
    B.pdf_xfxq2_members(h, 0, n_mem, pids, torch.from_numpy(xb).cuda(), torch.from_numpy(qb).cuda(), ob)
    torch.cuda.synchronize()
    assert B.pdf_grid_status(h) - before == 5
    bad = np.zeros(len(x), dtype=bool)
    bad[[3, 700, 2414, 9, 1000]] = True
    got = ob.cpu().numpy()
    assert np.isnan(got[:, :, bad]).all() and np.array_equal(got[:, :, ~bad], out.cpu().numpy()[:, :, ~bad])
    # a member range in the middle, a PID subset, the extrapolation mix (few jobs: persistent CTAs)
    xm, qm = W.queries_extrapolation_mix(g0, 20_011)
    sub = [21, -6, 2]
    dxm, dqm = torch.from_numpy(xm).cuda(), torch.from_numpy(qm).cuda()
    o2 = torch.empty((3, len(sub), len(xm)), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2_members(h, 7, 3, sub, dxm, dqm, o2)
    o1 = torch.empty((len(sub), len(xm)), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, sub, dxm, dqm, o1)
    torch.cuda.synchronize()
    r2, s2 = oracle.xfxq2_members(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals[7:10], sub, xm, qm, with_scale=True)
    check_parity(o2.cpu().numpy(), r2, s2, max_clause_frac=5e-3, what="member range 7..9")
    r0, s0 = oracle.xfxq2_members(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals[:1], sub, xm, qm, with_scale=True)
    check_parity(o1.cpu().numpy(), r0[0], s0[0], max_clause_frac=5e-3, what="pdf_xfxq2 = member 0")
    # argument errors
    with pytest.raises(B.PdfbError):
        B.pdf_xfxq2_members(h, n_mem - 1, 2, sub, dxm, dqm, o2)
    B.pdf_xfxq2_members(h, 0, 0, sub, dxm, dqm, o2)  # empty range: nothing to do
    B.pdf_grid_free(h)
    # a set on a tiny grid takes the read-only-cache kernel (member = blockIdx.y)
    from test_oracle_pins import make_spec, rand_knots
    rng = np.random.default_rng(5)
    xk = rand_knots(rng, 1e-4, 1.0, 3)
    subs = [rand_knots(rng, 1.5, 3.0, 2), rand_knots(rng, 3.0, 9.0, 5)]
    tv = np.stack([np.concatenate([rng.normal(size=(len(xk), len(q), 2)).reshape(-1) for q in subs]) for _ in range(4)])
    spec = make_spec(xk, subs, [1, 21], values=[np.zeros((len(xk), len(q), 2)) for q in subs])
    ht = B.pdf_set_load(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, tv)
    assert not B.pdf_grid_uses_smem_path(ht)
    xs, qs = W.scan_points(spec, per_cell=4)
    ot = torch.empty((3, 2, len(xs)), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2_members(ht, 1, 3, [21, 1], torch.from_numpy(xs).cuda(), torch.from_numpy(qs).cuda(), ot)
    torch.cuda.synchronize()
    rt, st = oracle.xfxq2_members(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, tv[1:4], [21, 1], xs, qs, with_scale=True)
    check_parity(ot.cpu().numpy(), rt, st, what="tiny member set")
    B.pdf_grid_free(ht)


def test_member_set_low_q2_rows_double_buffered(torch_cuda):
    """More jobs than SMs on a small batch whose Q^2 values sit in the FIRST intervals of the table: the
    set kernel stages rows 0.. twice (one copy per in-flight job), and the stencils of Q^2 intervals 0
    and 1 reach the row below row 0 with weight exactly 0 -- also in the second copy, where that row is
    not the block in front of the slice.  x includes the first x interval (knot -1 of a row = the tail
    of the row below).  Whatever is read there must be finite: every member equals the oracle, no NaN;
    under the poisoned build (-DPDFB_CHECKED) an unstaged read shows up as NaN."""
    torch = torch_cuda
    n_mem = 60                                   # 240 jobs > 148 SMs: persistent CTAs, next job's rows in flight
    g0 = W.grid_member(0)
    vals = W.member_values(n_mem)
    h = B.pdf_set_load(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals)
    assert B.pdf_grid_uses_smem_path(h)
    pids = list(W.PIDS_13)
    q2k = np.asarray(g0.q_knots[:4], dtype=np.float64) ** 2
    rng = np.random.Generator(np.random.PCG64(4242))
    n = 3001
    x = np.exp(rng.uniform(np.log(g0.x_knots[0]), np.log(g0.x_knots[-1]), n))
    x[:600] = np.exp(rng.uniform(np.log(g0.x_knots[0]), np.log(g0.x_knots[1]), 600))   # first x interval
    x[0], x[1] = g0.x_knots[0], g0.x_knots[1]
    x = np.clip(x, g0.x_knots[0], g0.x_knots[-1])
    cases = {
        "interval 1 only": np.exp(rng.uniform(np.log(q2k[1]), np.log(q2k[2]), n)).clip(q2k[1], q2k[2] * (1 - 1e-12)),
        "intervals 0 and 1": np.exp(rng.uniform(np.log(q2k[0]), np.log(q2k[2]), n)).clip(q2k[0], q2k[2] * (1 - 1e-12)),
        "interval 0 only": np.exp(rng.uniform(np.log(q2k[0]), np.log(q2k[1]), n)).clip(q2k[0], q2k[1] * (1 - 1e-12)),
        "intervals 1 and 2": np.exp(rng.uniform(np.log(q2k[1]), np.log(q2k[3]), n)).clip(q2k[1], q2k[3] * (1 - 1e-12)),
    }
    dx = torch.from_numpy(x).cuda()
    for name, q2 in cases.items():
        dq = torch.from_numpy(q2).cuda()
        out = torch.empty((n_mem, len(pids), n), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2_members(h, 0, n_mem, pids, dx, dq, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.isfinite(got).all(), name
        ref, sc = oracle.xfxq2_members(g0.x_knots, g0.q_offsets, g0.q_knots, g0.pids, vals, pids, x, q2, with_scale=True)
        check_parity(got, ref, sc, what="member set, low rows: " + name)
    B.pdf_grid_free(h)


def test_set_loaded_from_lhapdf_layout_files(torch_cuda, tmp_path):
    """A synthetic set written in the LHAPDF6 text layout (3 member files + metadata with the alpha_s
    nodes) and loaded through the front-end evaluates bit-identically to the same arrays loaded
    directly, and agrees with the oracle."""
    torch = torch_cuda
    d = tmp_path / "synthset"
    d.mkdir()
    pids = list(W.PIDS_13)
    specs = [W.grid_member(m) for m in range(3)]
    for m, sp in enumerate(specs):
        W.write_lhagrid(sp, str(d / f"synthset_{m:04d}.dat"), "central" if m == 0 else "replica")
    aspec = W.make_alphas_grid()
    W.write_lhapdf_info(str(d / "synthset.info"), 3, pids, aspec)
    hp, ha, fpids = B.load_lhapdf_set(str(d))
    assert B.pdf_set_members(hp) == 3 and list(fpids) == pids
    h_direct = B.pdf_set_load(specs[0].x_knots, specs[0].q_offsets, specs[0].q_knots, specs[0].pids,
                              np.stack([sp.values for sp in specs]))
    x, q2 = W.queries_extrapolation_mix(specs[0], 10_007)
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    o1 = torch.empty((3, len(pids), len(x)), dtype=torch.float64, device="cuda")
    o2 = torch.empty_like(o1)
    B.pdf_xfxq2_members(hp, 0, 3, pids, dx, dq, o1)
    B.pdf_xfxq2_members(h_direct, 0, 3, pids, dx, dq, o2)
    a1, a2 = torch.empty_like(dq), torch.empty_like(dq)
    B.alphas_q2(ha, dq, a1)
    hd = B.load_alphas_spec(aspec)
    B.alphas_q2(hd, dq, a2)
    torch.cuda.synchronize()
    assert torch.equal(o1, o2) and torch.equal(a1, a2)
    ref, sc = oracle.xfxq2_members(specs[0].x_knots, specs[0].q_offsets, specs[0].q_knots, specs[0].pids,
                                   [sp.values for sp in specs], pids, x, q2, with_scale=True)
    check_parity(o1.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what="set from files")
    for h in (hp, h_direct):
        B.pdf_grid_free(h)
    for h in (ha, hd):
        B.alphas_grid_free(h)


def test_pdf_object_api(torch_cuda, tmp_path):
    """mkPDF / PDF (Fig. 1): the four interpolating methods and the member form are
    single calls of the library -- same numbers as the binding calls, from a directory and from specs."""
    torch = torch_cuda
    from paper_2009_06635_b200 import PDF, mkPDF
    d = tmp_path / "objset"
    d.mkdir()
    specs = [W.grid_member(m) for m in range(2)]
    for m, sp in enumerate(specs):
        W.write_lhagrid(sp, str(d / f"objset_{m:04d}.dat"))
    aspec = W.make_alphas_grid()
    W.write_lhapdf_info(str(d / "objset.info"), 2, W.PIDS_13, aspec)
    x, q2 = W.queries_extrapolation_mix(specs[0], 5_003)
    q = np.sqrt(q2)
    with mkPDF(str(d)) as pdf, mkPDF(specs, alphas=aspec) as pdf2:
        assert isinstance(pdf, PDF) and pdf.n_members == 2 and pdf.pids == tuple(W.PIDS_13)
        a = pdf.xfxQ2([21, 1], x, q2)
        b = pdf2.xfxQ2([21, 1], torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda())
        assert a.shape == (2, len(x)) and torch.equal(a, b)
        ref, sc = oracle.OraclePdfGrid.from_spec(specs[0]).xfxq2([21, 1], x, q2, with_scale=True)
        check_parity(a.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what="PDF.xfxQ2")
        allm = pdf.xfxQ2(None, x, q2, members=(0, 2))
        assert allm.shape == (2, 13, len(x))
        # PID 21 is the last of PIDS_13 (2-column plan for the pair, 4-column plan for all 13: same
        # numbers up to summation order)
        assert torch.allclose(allm[0, 12], a[0], rtol=1e-11, atol=1e-14)
        assert torch.equal(pdf.xfxQ(None, x, q, members=(0, 2)), pdf.xfxQ2(None, x, q * q, members=(0, 2)))
        assert torch.equal(pdf.xfxQ([2], x, q), pdf.xfxQ2([2], x, q * q))
        al = pdf.alphasQ2(q2)
        check_parity(al.cpu().numpy(), oracle.OracleAlphas.from_spec(aspec).q2(q2), what="PDF.alphasQ2")
        assert torch.equal(pdf.alphasQ(q), pdf.alphasQ2(q * q)) and torch.equal(al, pdf2.alphasQ2(q2))
        assert pdf.n_invalid() == 0


def test_two_column_slices(torch_cuda, grid2, ograph2, monkeypatch):
    """The 2-column shared-memory path (row pairs as one 8-chunk run): (a) forced for every request
    on the NNPDF-shaped grid, (b) chosen by itself for one- and two-flavour requests, (c) the only
    shared-memory path of a grid whose 4-column slice does not fit (150 x 50 knots)."""
    torch = torch_cuda
    pids = list(W.PIDS_11)
    x, q2 = W.queries_extrapolation_mix(grid2, 40_003)
    xs, qs = W.scan_points(grid2, per_cell=2)
    x, q2 = np.concatenate([x, xs]), np.concatenate([q2, qs])
    ref, sc = ograph2.xfxq2(pids, x, q2, with_scale=True)
    monkeypatch.setenv("PDFB_NO_W4", "1")
    h = B.load_pdf_spec(grid2)
    monkeypatch.delenv("PDFB_NO_W4")
    assert B.pdf_grid_uses_smem_path(h)
    check_parity(gpu_xfxq2(torch, h, pids, x, q2), ref, sc, max_clause_frac=5e-3, what="2-column path, 11 flavours")
    sub = [21, 21, -5, 3]
    rs, ss = ograph2.xfxq2(sub, x, q2, with_scale=True)
    check_parity(gpu_xfxq2(torch, h, sub, x, q2), rs, ss, max_clause_frac=5e-3, what="2-column path, duplicates")
    B.pdf_grid_free(h)
    # (b) default handle: narrow requests take the 2-column plan, same numbers within tolerance
    h = B.load_pdf_spec(grid2)
    for req in ([21], [4, 5], [-5]):
        r1, s1 = ograph2.xfxq2(req, x, q2, with_scale=True)
        check_parity(gpu_xfxq2(torch, h, req, x, q2), r1, s1, max_clause_frac=5e-3, what=f"narrow request {req}")
    B.pdf_grid_free(h)
    # (c) a grid too large for 4-column slices
    big = W.make_pdf_grid(1e-9, 1.0, 150, (1.65, 4.92, 172.5, 1.0e5), (10, 20, 20), W.PIDS_11)
    hb = B.load_pdf_spec(big)
    assert B.pdf_grid_uses_smem_path(hb)
    xb, qb = W.queries_extrapolation_mix(big, 30_011)
    xs, qs = W.scan_points(big, per_cell=1)
    xb, qb = np.concatenate([xb, xs]), np.concatenate([qb, qs])
    rb, sb = oracle.OraclePdfGrid.from_spec(big).xfxq2(pids, xb, qb, with_scale=True)
    check_parity(gpu_xfxq2(torch, hb, pids, xb, qb), rb, sb, max_clause_frac=5e-3, what="150 x 50 grid")
    B.pdf_grid_free(hb)
