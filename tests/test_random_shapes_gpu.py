"""GPU parity over RANDOM grid shapes (seeded): number of x knots, number and length of the Q^2
sub-grids, number of flavours and knot spacing are drawn per case, so that every layout decision of
the library is hit by some case -- 4-column slices, 2-column slices only, the read-only-cache kernel
(fewer than 4 knots somewhere), nx not a multiple of 4, one to five sub-grids, 1 to 14 PIDs, partly
filled flavour groups -- on the calls pdf_xfxq2, pdf_xfxq2_pm and pdf_lumi_events.  Every cell, knot
and threshold of each grid is scanned and a mix of points outside the grid is added."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2009_06635_b200 import binding as B, build, workloads as W
from parity_util import check_parity

PID_POOL = (-6, -5, -4, -3, -2, -1, 1, 2, 3, 4, 5, 6, 21, 22)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    build.build()
    B.lib()
    return torch


def jittered_knots(rng, lo, hi, n, jitter):
    """Log-spaced knots, the interior ones moved by up to +-jitter of a spacing (ln gaps stay >= (1 - 2 jitter) of it)."""
    z = np.linspace(np.log(lo), np.log(hi), n)
    if n > 2:
        z[1:-1] += rng.uniform(-jitter, jitter, n - 2) * (z[1] - z[0])
    k = np.exp(z)
    k[0], k[-1] = lo, hi
    return k


def random_spec(rng):
    nx = int(rng.choice([2, 3, 4, 5, 7, 13, 30, 61, 100, 118, 150]))
    n_sub = int(rng.integers(1, 6))
    nq = [int(rng.choice([2, 3, 4, 5, 6, 9, 14, 25])) for _ in range(n_sub)]
    n_pid = int(rng.integers(1, 15))
    pids = [int(p) for p in rng.choice(PID_POOL, size=n_pid, replace=False)]
    jitter = float(rng.choice([0.0, 0.15, 0.3]))
    x_lo = float(10.0 ** rng.uniform(-9, -3))
    edges = np.exp(np.linspace(np.log(1.3), np.log(float(10.0 ** rng.uniform(2, 5))), n_sub + 1))
    xk = jittered_knots(rng, x_lo, 1.0, nx, jitter)
    params = W.draw_family_params(pids, int(rng.integers(1, 1 << 30)))
    q_knots, offs, vals = [], [0], []
    for s in range(n_sub):
        q = jittered_knots(rng, float(edges[s]), float(edges[s + 1]), nq[s], jitter)
        q_knots.append(q)
        offs.append(offs[-1] + nq[s])
        blk = np.stack([W.family_value(params[p], xk[:, None], (q * q)[None, :]) for p in pids], axis=-1)
        vals.append(blk.reshape(-1))
    return W.PdfGridSpec(xk, np.asarray(offs, np.int32), np.concatenate(q_knots), np.asarray(pids, np.int32),
                         np.concatenate(vals), params)


COORD_ULPS = 4   # see coord_slack


def near_one(spec, x):
    """The points a coarse x array makes ill-conditioned in t (see coord_slack)."""
    x = np.asarray(x)
    return (x > 0.99) & (x < 1.0) if spec.nx < 8 else np.zeros(x.shape, dtype=bool)


def coord_slack(spec, xfx, x, q2):
    """Extra |d| allowed at points just below x = 1 on an x array of fewer than 8 knots; zero elsewhere.

    There the last interval spans orders of magnitude in x while xf falls to exactly 0 at x = 1, so the
    result is (1 - t) * slope: a difference of nearly equal terms in the in-cell coordinate t itself.  The
    library forms t = (u - z0) * (1/dz) where the oracle divides, (u - z0) / dz: the reciprocal and the
    product round twice where the division rounds once, so the two t differ by up to 3 * 2^-53 on t ~ 1
    (the difference u - z0 rounds the same way on both sides).  That moves the result by |d ref / d t|
    times 3 * 2^-53 whatever 1 - t is -- relative to the RESULT it is 1e-16 / (1 - t), beyond the 1e-12 rule
    once 1 - t < 1e-4, for the oracle against exact arithmetic as much as for the library against the
    oracle.  (With the >= 30 knots of real grids such results are far below 1e-3 and the absolute rule
    applies.)  So these points are checked against
        |d| <= rule(ref) + COORD_ULPS * 2^-53 * |d ref / d t|,        COORD_ULPS = 4,
    d ref / d t = dz * d ref / d ln x from a one-sided finite difference of the oracle (h = 1e-6, towards
    smaller x: the same interval).  A wrong cell, weight or table entry is off by ~|slope| itself, 1e15 times
    the allowance.  Measured on the 44 seeded cases (B200): 4 outputs need it, at most 0.52 of it (the
    parity summary at the end of a run prints the uses).  ``xfx(x, q2)`` -> oracle values [..., n]."""
    m = near_one(spec, x)
    if not m.any():
        return None
    h = 1e-6
    dz = float(np.log(spec.x_knots[-1] / spec.x_knots[-2]))
    f0, f1 = xfx(x[m], q2[m]), xfx(x[m] * (1.0 - h), q2[m])
    slack = np.zeros(f0.shape[:-1] + (len(x),))
    slack[..., m] = COORD_ULPS * 2.0 ** -53 * dz * np.abs(f0 - f1) / h
    return slack


def points(rng, spec, n_out=1500):
    x, q2 = W.scan_points(spec, per_cell=1)
    if len(x) > 6000:  # large grids: a random subset of the scan
        keep = rng.choice(len(x), 6000, replace=False)
        x, q2 = x[keep], q2[keep]
    x_lo = float(spec.x_knots[0])
    xo = np.exp(rng.uniform(np.log(x_lo) - 4.0, 0.0, n_out))
    qo = np.exp(rng.uniform(np.log(spec.q2_min) - 1.5, np.log(spec.q2_max) + 1.5, n_out))
    return np.concatenate([x, xo]), np.concatenate([q2, qo])


@pytest.mark.parametrize("case", range(24))
def test_random_grid_shape(torch_cuda, case):
    torch = torch_cuda
    rng = np.random.default_rng(20090 + case)
    spec = random_spec(rng)
    og = oracle.OraclePdfGrid.from_spec(spec)
    h = B.load_pdf_spec(spec)
    shape = (spec.nx, [len(spec.sub_q(s)) for s in range(spec.n_sub)], spec.n_pid, bool(B.pdf_grid_uses_smem_path(h)))
    x, q2 = points(rng, spec)
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    pids = [int(p) for p in spec.pids]
    reqs = [pids, [pids[int(rng.integers(len(pids)))]]]
    if len(pids) > 2:
        reqs.append([int(p) for p in rng.choice(pids, size=min(len(pids), 5), replace=False)])
    for req in reqs:
        ref, sc = og.xfxq2(req, x, q2, with_scale=True)
        out = torch.full((len(req), len(x)), 7.0, dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h, req, dx, dq, out)
        pm = torch.full((len(x), len(req)), 7.0, dtype=torch.float64, device="cuda")
        B.pdf_xfxq2_pm(h, req, dx, dq, pm)
        torch.cuda.synchronize()
        st = check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"random shape {case} {shape} F={len(req)}", log=(req is pids),
                          slack=coord_slack(spec, lambda a, b: og.xfxq2(req, a, b), x, q2))
        # the point-major variant: the same numbers, transposed, bit for bit
        assert torch.equal(pm.t().contiguous().view(torch.int64), out.view(torch.int64)), shape
    # every knot reproduces its table value bit for bit -- the last knot of either axis included (t = 1 there
    # would come out of a rounded product; the library gives the last knot an interval of its own)
    for sg in range(spec.n_sub):
        q2k = spec.sub_q(sg) ** 2
        if sg + 1 < spec.n_sub:
            q2k = q2k[:-1]  # a threshold belongs to the upper sub-grid
        X, Q = np.meshgrid(spec.x_knots, q2k, indexing="ij")
        out = torch.empty((len(pids), X.size), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h, pids, torch.from_numpy(X.ravel().copy()).cuda(), torch.from_numpy(Q.ravel().copy()).cuda(), out)
        torch.cuda.synchronize()
        want = spec.sub_values(sg)[:, : len(q2k), :].transpose(2, 0, 1).reshape(len(pids), -1)
        assert np.array_equal(out.cpu().numpy(), want), (shape, sg)
    # the fused luminosity of events on the same grid (in range and outside), random signed coefficients
    n_ev = 3000
    x1 = np.exp(rng.uniform(np.log(float(spec.x_knots[0])) - 1.0, 0.0, n_ev))
    x2 = np.exp(rng.uniform(np.log(float(spec.x_knots[0])) - 1.0, 0.0, n_ev))
    qe = np.exp(rng.uniform(np.log(spec.q2_min) - 0.5, np.log(spec.q2_max) + 0.5, n_ev))
    terms = [(a, b, float(rng.normal())) for a in pids for b in pids if rng.uniform() < 0.4] or [(pids[0], pids[0], 1.0)]
    lum = torch.full((n_ev,), 7.0, dtype=torch.float64, device="cuda")
    B.pdf_lumi_events(h, terms, torch.from_numpy(x1).cuda(), torch.from_numpy(x2).cuda(), torch.from_numpy(qe).cuda(), lum)
    torch.cuda.synchronize()
    rl, sl = oracle.lumi_events(og, terms, x1, x2, qe, with_scale=True)
    # the luminosity's allowance at events with a beam just below x = 1 on a coarse x array: first order in
    # the factors' own allowances, sum_t |c_t| (slack_a(x1) |xf_b(x2)| + |xf_a(x1)| slack_b(x2))
    lslack = None
    if near_one(spec, x1).any() or near_one(spec, x2).any():
        f1, f2 = og.xfxq2(pids, x1, qe), og.xfxq2(pids, x2, qe)
        s1 = coord_slack(spec, lambda a, b: og.xfxq2(pids, a, b), x1, qe)
        s2 = coord_slack(spec, lambda a, b: og.xfxq2(pids, a, b), x2, qe)
        s1 = np.zeros_like(f1) if s1 is None else s1
        s2 = np.zeros_like(f2) if s2 is None else s2
        lslack = np.zeros(n_ev)
        for a, b, c in terms:
            ia, ib = pids.index(a), pids.index(b)
            lslack += abs(c) * (s1[ia] * np.abs(f2[ib]) + np.abs(f1[ia]) * s2[ib] + s1[ia] * s2[ib])
    check_parity(lum.cpu().numpy(), rl, sl, max_clause_frac=2e-2, what=f"random shape {case} lumi", log=False, slack=lslack)
    print("case", case, shape, st)
    B.pdf_grid_free(h)


@pytest.mark.parametrize("case", range(16))
def test_random_alphas_node_lists(torch_cuda, case):
    """alpha_s on random node lists: 2 to 512 nodes (the replicated-line fast path up to 192, the general
    kernel beyond), one to five sub-grids split by repeated nodes, sub-grids of two nodes, jittered
    spacing, values from one-loop running times a random smooth factor.  Queries: every node, its two
    neighbouring doubles, points inside every interval, outside the list, invalid scales; alphas_q as well."""
    torch = torch_cuda
    rng = np.random.default_rng(7300 + case)
    n_sub = int(rng.integers(1, 6))
    total = int(rng.choice([2, 3, 5, 17, 60, 100, 191, 192, 193, 300, 512]))
    total = max(total, 2 * n_sub)
    cuts = np.sort(rng.choice(np.arange(1, total - 1), size=n_sub - 1, replace=False)) if n_sub > 1 and total > 2 * n_sub else \
        np.arange(2, 2 * n_sub, 2)[: n_sub - 1]
    sizes = np.diff(np.concatenate([[0], cuts, [total]])).astype(int)
    sizes = np.maximum(sizes, 2)
    edges = np.exp(np.linspace(np.log(1.0), np.log(float(10.0 ** rng.uniform(2, 5))), n_sub + 1))
    jitter = float(rng.choice([0.0, 0.2, 0.35]))
    qs, al = [], []
    for s in range(n_sub):
        q = jittered_knots(rng, float(edges[s]), float(edges[s + 1]), int(sizes[s]), jitter)
        a = W.one_loop_alphas(q * q) * (1.0 + 0.05 * s + 0.02 * np.sin(np.log(q)))
        qs.append(q); al.append(a)
    spec = W.AlphasSpec(np.concatenate(qs), np.concatenate(al))
    if len(spec.q_knots) > 512:
        pytest.skip("more than 512 nodes after padding the sub-grids")
    oa = oracle.OracleAlphas.from_spec(spec)
    ha = B.load_alphas_spec(spec)
    k2 = spec.q_knots ** 2
    mids = [np.sqrt(k2[:-1] * k2[1:]), k2[:-1] ** 0.9 * k2[1:] ** 0.1, k2[:-1] ** 0.1 * k2[1:] ** 0.9]
    q2 = np.concatenate([k2, np.nextafter(k2, 0), np.nextafter(k2, np.inf)] + mids +
                        [np.exp(rng.uniform(np.log(k2[0]) - 3, np.log(k2[-1]) + 3, 3000)), [0.0, -2.0, np.nan, np.inf]])
    dq = torch.from_numpy(q2).cuda()
    out = torch.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    dq1 = torch.from_numpy(np.sqrt(np.where(q2 > 0, q2, np.nan))).cuda()
    out1 = torch.empty_like(dq1)
    B.alphas_q(ha, dq1, out1)
    torch.cuda.synchronize()
    ref = oa.q2(q2)
    check_parity(out.cpu().numpy(), ref, what=f"random alpha_s list {case}: {len(k2)} nodes, sub-grids {list(sizes)}", log=False)
    # alphas_q(Q) is alphas_q2 at Q*Q rounded once: compare with the oracle at that argument
    qq = dq1.cpu().numpy()
    ref1 = oa.q2(np.where(np.isnan(qq), -1.0, qq * qq))
    check_parity(out1.cpu().numpy(), ref1, what=f"random alpha_s list {case}, Q argument", log=False)
    B.alphas_grid_free(ha)


@pytest.mark.parametrize("case", range(12))
def test_random_member_sets(torch_cuda, case):
    """PDF sets on random grid shapes: 2 to 60 members (fewer and more (member, flavour group) jobs than
    SMs), a small batch at one scale (rows of the batch's Q^2 range only, the points' cell and t cached in
    shared memory), a small batch over the whole Q^2 range with points outside the grid and on the last
    knots, and a batch too large for either; member ranges; the Q-argument entry point."""
    torch = torch_cuda
    rng = np.random.default_rng(9100 + case)
    spec = random_spec(rng)
    n_mem = int(rng.choice([2, 5, 13, 40, 60]))
    vals = np.stack([spec.values * (1.0 + 0.3 * rng.normal()) + 0.01 * rng.normal(size=spec.values.shape) * np.abs(spec.values)
                     for _ in range(n_mem)])
    h = B.pdf_set_load(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, vals)
    pids = [int(p) for p in spec.pids]
    x_lo = float(spec.x_knots[0])
    q_one = float(np.exp(rng.uniform(np.log(spec.q2_min), np.log(spec.q2_max))))
    batches = {
        "one scale": (np.exp(rng.uniform(np.log(x_lo), 0.0, 1203)), np.full(1203, q_one)),
        "top of the grid": (np.concatenate([np.exp(rng.uniform(np.log(x_lo), 0.0, 700)), [1.0, 1.0, x_lo]]),
                            np.concatenate([np.full(700, spec.q2_max), [spec.q2_max, q_one, spec.q2_max]])),
        "mix": points(rng, spec, n_out=800),
        "large": (np.exp(rng.uniform(np.log(x_lo) - 1.0, 0.0, 70_001)),
                  np.exp(rng.uniform(np.log(spec.q2_min) - 0.3, np.log(spec.q2_max) + 0.3, 70_001))),
    }
    for name, (x, q2) in batches.items():
        m0 = int(rng.integers(0, n_mem))
        cnt = int(rng.integers(1, n_mem - m0 + 1)) if name != "large" else min(2, n_mem - m0)
        req = pids if name != "large" else pids[: min(len(pids), 5)]
        dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
        out = torch.full((cnt, len(req), len(x)), 7.0, dtype=torch.float64, device="cuda")
        B.pdf_xfxq2_members(h, m0, cnt, req, dx, dq, out)
        outq = torch.full_like(out, 7.0)
        B.pdf_xfxq2_members(h, m0, cnt, req, dx, torch.sqrt(dq), outq, q_is_q=True)
        torch.cuda.synchronize()
        members = lambda a, b: oracle.xfxq2_members(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, vals[m0:m0 + cnt], req, a, b)
        ref, sc = oracle.xfxq2_members(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, vals[m0:m0 + cnt], req, x, q2, with_scale=True)
        check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"random set {case} {name}: {n_mem} members, range {m0}+{cnt}", log=False,
                     slack=coord_slack(spec, members, x, q2))
        q2r = np.sqrt(q2) ** 2  # what the Q-argument call evaluates at: Q*Q rounded once
        refq, scq = oracle.xfxq2_members(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, vals[m0:m0 + cnt], req, x, q2r, with_scale=True)
        check_parity(outq.cpu().numpy(), refq, scq, max_clause_frac=5e-3, what=f"random set {case} {name}, Q argument", log=False,
                     slack=coord_slack(spec, members, x, q2r))
    B.pdf_grid_free(h)


@pytest.mark.parametrize("case", range(8))
def test_random_per_subgrid_x_knots_files_and_variants(torch_cuda, case, tmp_path):
    """Sub-grids with their own x-knot arrays (different lengths and spacings on one [x_min, x_max]) on random
    shapes, loaded directly and through a member file in the LHAPDF text layout; on the same handle the
    fp32-output variant (= the fp64 result rounded once) and the host-buffer entry point (= the device call)."""
    torch = torch_cuda
    rng = np.random.default_rng(5500 + case)
    n_sub = int(rng.integers(2, 5))
    nq = [int(rng.choice([2, 4, 6, 11])) for _ in range(n_sub)]
    n_pid = int(rng.integers(1, 12))
    pids = [int(p) for p in rng.choice(PID_POOL, size=n_pid, replace=False)]
    x_lo = float(10.0 ** rng.uniform(-8, -3))
    xs = [jittered_knots(rng, x_lo, 1.0, int(rng.choice([4, 9, 26, 60, 97])), float(rng.choice([0.0, 0.3]))) for _ in range(n_sub)]
    edges = tuple(float(e) for e in np.exp(np.linspace(np.log(1.4), np.log(3e3), n_sub + 1)))
    spec = W.make_pdf_grid_xs(xs, edges, tuple(nq), pids, seed=int(rng.integers(1, 1 << 30)))
    og = oracle.OraclePdfGrid.from_spec(spec)
    h = B.load_pdf_spec(spec)
    n = 4001
    x = np.exp(rng.uniform(np.log(x_lo) - 2.0, 0.0, n))
    q2 = np.exp(rng.uniform(np.log(spec.q2_min) - 1.0, np.log(spec.q2_max) + 1.0, n))
    x[:3], q2[:3] = [1.0, x_lo, 1.0], [spec.q2_max, spec.q2_max, spec.q2_min]
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    out = torch.empty((n_pid, n), dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, pids, dx, dq, out)
    o32 = torch.empty((n_pid, n), dtype=torch.float32, device="cuda")
    B.pdf_xfxq2_f32(h, pids, dx, dq, o32)
    torch.cuda.synchronize()
    ref, sc = og.xfxq2(pids, x, q2, with_scale=True)
    check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"random per-sub-grid x knots {case}", log=False)
    assert torch.equal(o32, out.to(torch.float32))
    host = np.empty((n_pid, n))
    B.pdf_xfxq2_host(h, pids, x, q2, host)
    assert np.array_equal(host, out.cpu().numpy(), equal_nan=True)
    for s in range(spec.n_sub):   # every knot of every sub-grid, bit for bit
        q = spec.sub_q(s) if s + 1 == spec.n_sub else spec.sub_q(s)[:-1]
        X, Q = np.meshgrid(spec.sub_x(s), q ** 2, indexing="ij")
        ok = torch.empty((n_pid, X.size), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h, pids, torch.from_numpy(X.ravel().copy()).cuda(), torch.from_numpy(Q.ravel().copy()).cuda(), ok)
        torch.cuda.synchronize()
        assert np.array_equal(ok.cpu().numpy(), spec.sub_values(s)[:, :len(q), :].transpose(2, 0, 1).reshape(n_pid, -1)), s
    d = tmp_path / "rset"
    d.mkdir()
    W.write_lhagrid(spec, str(d / "rset_0000.dat"))
    W.write_lhapdf_info(str(d / "rset.info"), 1, pids, W.make_alphas_grid())
    hf, ha, fp = B.load_lhapdf_set(str(d))
    of = torch.empty_like(out)
    B.pdf_xfxq2(hf, pids, dx, dq, of)
    torch.cuda.synchronize()
    assert list(fp) == pids and torch.equal(of.view(torch.int64), out.view(torch.int64))
    B.pdf_grid_free(hf); B.alphas_grid_free(ha); B.pdf_grid_free(h)


@pytest.mark.parametrize("case", range(8))
def test_random_large_mixes(torch_cuda, case):
    """Many tiles per CTA on random shapes, with the out-of-grid share of the batch anywhere between 0 and 95 %
    and any split between the five continuation classes: the class lists fill, trigger and flush at every
    rhythm (a list reaching the trigger in one tile, lists that never do, all classes at once)."""
    torch = torch_cuda
    rng = np.random.default_rng(6600 + case)
    while True:  # a shape the shared-memory kernel takes (every sub-grid has at least 4 Q^2 knots)
        spec = random_spec(rng)
        if spec.nx >= 8 and min(len(spec.sub_q(s)) for s in range(spec.n_sub)) >= 4:
            break
    og = oracle.OraclePdfGrid.from_spec(spec)
    h = B.load_pdf_spec(spec)
    assert B.pdf_grid_uses_smem_path(h)
    pids = [int(p) for p in spec.pids]
    n = 400_003
    f_out = float(rng.choice([0.0, 0.02, 0.3, 0.7, 0.95]))
    lx0, lq0, lq1 = np.log(float(spec.x_knots[0])), np.log(spec.q2_min), np.log(spec.q2_max)
    x = np.exp(rng.uniform(lx0, 0.0, n))
    q2 = np.exp(rng.uniform(lq0, lq1, n))
    out_pts = rng.uniform(size=n) < f_out
    p_cls = rng.dirichlet(np.ones(3))                      # low x | high Q | low Q (corners where two coincide)
    kind = rng.choice(3, size=n, p=p_cls)
    both = rng.uniform(size=n) < 0.2
    low_x = out_pts & ((kind == 0) | both)
    high_q = out_pts & (kind == 1)
    low_q = out_pts & (kind == 2)
    x[low_x] = np.exp(rng.uniform(lx0 - 6.0, lx0, int(low_x.sum())))
    q2[high_q] = np.exp(rng.uniform(lq1, lq1 + 3.0, int(high_q.sum())))
    q2[low_q] = np.exp(rng.uniform(lq0 - 2.0, lq0, int(low_q.sum())))
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    out = torch.full((len(pids), n), 7.0, dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h, pids, dx, dq, out)
    again = torch.full_like(out, 7.0)
    B.pdf_xfxq2(h, pids, dx, dq, again)
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int64), again.view(torch.int64))
    ref, sc = og.xfxq2(pids, x, q2, with_scale=True)
    st = check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=1e-2,
                      what=f"random large mix {case}: nx {spec.nx}, {spec.n_pid} PIDs, {f_out:.0%} outside", log=False)
    print("\ncase", case, spec.nx, [len(spec.sub_q(s)) for s in range(spec.n_sub)], spec.n_pid, f_out, st)
    B.pdf_grid_free(h)
