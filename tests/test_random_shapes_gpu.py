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
        st = check_parity(out.cpu().numpy(), ref, sc, max_clause_frac=5e-3, what=f"random shape {case} {shape} F={len(req)}", log=(req is pids))
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
    check_parity(lum.cpu().numpy(), rl, sl, max_clause_frac=2e-2, what=f"random shape {case} lumi", log=False)
    print("case", case, shape, st)
    B.pdf_grid_free(h)
