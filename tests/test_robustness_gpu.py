"""GPU checks of what DESIGN.md promises about a handle in use, beyond element-wise parity:
several streams evaluating on ONE handle at the same time (the per-SM scratch of the out-of-grid
class lists, the row-range slots of small batches), bit-identical results run to run, and batch
sizes around every granularity of the launch (a warp, a tile, the row-range threshold)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2009_06635_b200 import binding as B, build, workloads as W
from parity_util import check_parity


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    build.build()
    B.lib()
    return torch


@pytest.fixture(scope="module")
def h2(torch_cuda, grid2):
    h = B.load_pdf_spec(grid2)
    yield h
    B.pdf_grid_free(h)


def test_streams_share_one_handle(torch_cuda, grid2, ograph2, h2):
    """Four streams, each with its own extrapolation-mix batch (30 % of the points go through the
    class lists in the handle's scratch), all in flight on one handle, several rounds: every result
    equals the one the same batch gives alone, bit for bit, and agrees with the oracle."""
    torch = torch_cuda
    pids = list(W.PIDS_11)
    n = 400_003
    batches = []
    for k in range(4):
        x, q2 = W.queries_extrapolation_mix(grid2, n, config=7000 + k)
        batches.append((torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), x, q2))
    alone = []
    for dx, dq, _, _ in batches:
        out = torch.empty((len(pids), n), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h2, pids, dx, dq, out)
        torch.cuda.synchronize()
        alone.append(out)
    streams = [torch.cuda.Stream() for _ in batches]
    outs = [torch.empty((len(pids), n), dtype=torch.float64, device="cuda") for _ in batches]
    for rnd in range(5):
        for o in outs:
            o.fill_(float("nan"))
        torch.cuda.synchronize()
        for (dx, dq, _, _), s, o in zip(batches, streams, outs):
            B.pdf_xfxq2(h2, pids, dx, dq, o, stream=s)
        torch.cuda.synchronize()
        for k, (o, a) in enumerate(zip(outs, alone)):
            assert torch.equal(o.view(torch.int64), a.view(torch.int64)), (rnd, k)
    _, _, x, q2 = batches[0]
    ref, sc = ograph2.xfxq2(pids, x[:50_000], q2[:50_000], with_scale=True)
    check_parity(alone[0][:, :50_000].cpu().numpy(), ref, sc, max_clause_frac=5e-3, what="streams")
    assert B.pdf_grid_status(h2) == 0


def test_small_batches_in_flight_share_the_row_range_slots(torch_cuda, grid2, ograph2, h2):
    """Small batches (<= 65 536 points) first find the table rows they touch and take one of the
    handle's slots for it: 24 such calls in flight on three streams, each on a different Q^2 band."""
    torch = torch_cuda
    pids = [21, 1, -2]
    rng = np.random.default_rng(99)
    q_lo, q_hi = np.log(grid2.q2_min), np.log(grid2.q2_max)
    streams = [torch.cuda.Stream() for _ in range(3)]
    jobs = []
    for k in range(24):
        n = int(rng.integers(1, 6000))
        a = q_lo + (q_hi - q_lo) * rng.uniform(0, 0.9)
        b = min(q_hi, a + (q_hi - q_lo) * rng.uniform(0.0, 0.1))
        x = np.exp(rng.uniform(np.log(grid2.x_knots[0]), 0.0, n))
        q2 = np.clip(np.exp(rng.uniform(a, b, n)), grid2.q2_min, grid2.q2_max)
        out = torch.empty((len(pids), n), dtype=torch.float64, device="cuda")
        jobs.append((x, q2, torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda(), out))
    for k, (_, _, dx, dq, out) in enumerate(jobs):
        B.pdf_xfxq2(h2, pids, dx, dq, out, stream=streams[k % 3])
    torch.cuda.synchronize()
    for x, q2, _, _, out in jobs:
        ref, sc = ograph2.xfxq2(pids, x, q2, with_scale=True)
        check_parity(out.cpu().numpy(), ref, sc, what="row-range slots", log=False)


def test_bit_identical_run_to_run(torch_cuda, grid2, h2):
    """a given batch is bit-reproducible run to run, out-of-grid points included
    (batch k of a class list is always the warp's entries 32k .. 32k+31, whenever it runs)."""
    torch = torch_cuda
    pids = list(W.PIDS_11)
    x, q2 = W.queries_extrapolation_mix(grid2, 1_000_003)
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    first = None
    for _ in range(4):
        out = torch.full((len(pids), len(x)), float("nan"), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h2, pids, dx, dq, out)
        torch.cuda.synchronize()
        if first is None:
            first = out
        else:
            assert torch.equal(out.view(torch.int64), first.view(torch.int64))


@pytest.mark.parametrize("pids", [[21], [2, -2, 21, 5, 1]])
def test_ragged_sizes(torch_cuda, grid2, ograph2, h2, pids):
    """Sizes around a warp, a tile of 512, one tile per SM, and the small-batch threshold; the tail
    of every batch holds out-of-grid points (their lists are flushed at the end of the launch).
    A launch on n points leaves the rest of a longer output buffer alone."""
    torch = torch_cuda
    x, q2 = W.queries_extrapolation_mix(grid2, 80_000, config=31)
    dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
    ref, sc = ograph2.xfxq2(pids, x, q2, with_scale=True)
    for n in (1, 2, 31, 32, 33, 511, 512, 513, 1023, 75_263, 75_264, 75_265, 65_535, 65_536, 65_537, 80_000):
        dense = torch.empty((len(pids), n), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h2, pids, dx, dq, dense, n=n)
        torch.cuda.synchronize()
        got = dense.cpu().numpy()
        check_parity(got, ref[:, :n], sc[:, :n], max_clause_frac=1.0 if n < 2000 else 5e-3, what=f"ragged n={n}", log=False)
    # the guard: a launch on n points leaves the rest of a larger buffer alone
    n = 70_001
    big = torch.full((len(pids) * n + 4096,), -7.0, dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h2, pids, dx, dq, big, n=n)
    torch.cuda.synchronize()
    assert bool((big[len(pids) * n:] == -7.0).all())


def test_calls_can_be_captured_in_a_cuda_graph(torch_cuda, grid2, ograph2, h2):
    """include/pdfb200.h: the evaluation calls allocate nothing and never synchronise.  A launch-bound
    loop can therefore be captured once and replayed: pdf_xfxq2 (a small batch, which also runs the
    row-range pre-pass), pdf_xfxq2 on an extrapolation mix, alphas_q2 and pdf_lumi_events in ONE graph;
    after the inputs are overwritten in place, a replay gives bit for bit what direct calls give."""
    torch = torch_cuda
    pids = list(W.PIDS_11)
    aspec = W.make_alphas_grid()
    ha = B.load_alphas_spec(aspec)
    n_s, n_m = 3_001, 150_001
    terms = [(1, -1, 1.0), (-2, 2, 0.5), (21, 21, 0.25)]

    def inputs(k):
        xs, qs = W.queries_in_range(grid2, n_s, 40 + k)
        xm, qm = W.queries_extrapolation_mix(grid2, n_m, config=50 + k)
        x1, x2, qe = W.queries_mc_events(grid2, n_m, config=60 + k)
        return [torch.from_numpy(a).cuda() for a in (xs, qs, xm, qm, x1, x2, qe)]

    buf = inputs(0)
    xs, qs, xm, qm, x1, x2, qe = buf
    o_s = torch.empty((len(pids), n_s), dtype=torch.float64, device="cuda")
    o_m = torch.empty((len(pids), n_m), dtype=torch.float64, device="cuda")
    o_a = torch.empty(n_m, dtype=torch.float64, device="cuda")
    o_l = torch.empty(n_m, dtype=torch.float64, device="cuda")

    def calls(os_, om_, oa_, ol_):
        B.pdf_xfxq2(h2, pids, xs, qs, os_)
        B.pdf_xfxq2(h2, pids, xm, qm, om_)
        B.alphas_q2(ha, qe, oa_)
        B.pdf_lumi_events(h2, terms, x1, x2, qe, ol_)

    calls(o_s, o_m, o_a, o_l)  # first use outside the capture (function attributes are set on first use)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        calls(o_s, o_m, o_a, o_l)
    for k in (1, 2):
        for dst, src in zip(buf, inputs(k)):
            dst.copy_(src)
        for o in (o_s, o_m, o_a, o_l):
            o.fill_(float("nan"))
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        d = [torch.empty_like(o) for o in (o_s, o_m, o_a, o_l)]
        calls(*d)
        torch.cuda.synchronize()
        for got, want in zip((o_s, o_m, o_a, o_l), d):
            assert torch.equal(got.view(torch.int64), want.view(torch.int64)), k
    ref, sc = ograph2.xfxq2(pids, xs.cpu().numpy(), qs.cpu().numpy(), with_scale=True)
    check_parity(o_s.cpu().numpy(), ref, sc, what="graph replay, small batch")
    B.alphas_grid_free(ha)


def test_graph_replay_next_to_live_small_batches(torch_cuda, grid2, h2):
    """A small batch first asks a one-CTA pre-pass which table rows it needs; the answer sits in a
    per-handle slot.  A call recorded into a CUDA graph keeps its slot for every replay, so recorded calls
    take theirs from a ring that live calls never use (xfxq2_smem.cu): a graph replaying on one stream
    while hundreds of live small batches -- on other table rows -- go through the live ring on another
    stream still gives, bit for bit, what the same call gives alone; so does every live call."""
    torch = torch_cuda
    pids = list(W.PIDS_11)
    n_s = 2_003
    rng = np.random.Generator(np.random.PCG64(99))
    q2k = np.asarray(grid2.q_knots, dtype=np.float64) ** 2
    x = np.exp(rng.uniform(np.log(grid2.x_knots[0]), np.log(grid2.x_knots[-1]), n_s)).clip(grid2.x_knots[0], grid2.x_knots[-1])
    q_lo = np.exp(rng.uniform(np.log(q2k[1]), np.log(q2k[3]), n_s)).clip(q2k[1], q2k[3])          # bottom rows
    q_hi = np.exp(rng.uniform(np.log(q2k[-4]), np.log(q2k[-2]), n_s)).clip(q2k[-4], q2k[-2])      # top rows
    dx, dlo, dhi = (torch.from_numpy(a).cuda() for a in (x, q_lo, q_hi))
    want_lo = torch.empty((len(pids), n_s), dtype=torch.float64, device="cuda")
    want_hi = torch.empty_like(want_lo)
    B.pdf_xfxq2(h2, pids, dx, dlo, want_lo)
    B.pdf_xfxq2(h2, pids, dx, dhi, want_hi)
    torch.cuda.synchronize()
    side, live = torch.cuda.Stream(), torch.cuda.Stream()
    o_g = torch.empty_like(want_lo)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        B.pdf_xfxq2(h2, pids, dx, dlo, o_g)
    n_live = 40
    o_live = [torch.empty_like(want_hi) for _ in range(n_live)]
    for rnd in range(12):                          # 480 live calls: the live ring wraps seven times
        o_g.fill_(float("nan"))
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            for _ in range(20):
                graph.replay()
        for o in o_live:
            B.pdf_xfxq2(h2, pids, dx, dhi, o, stream=live)
        torch.cuda.synchronize()
        assert torch.equal(o_g.view(torch.int64), want_lo.view(torch.int64)), rnd
        for o in o_live:
            assert torch.equal(o.view(torch.int64), want_hi.view(torch.int64)), rnd


def test_more_than_2_to_the_31_points(torch_cuda, grid2, ograph2, h2):
    """Maximum sizes: the class lists hold point indices as 32-bit offsets, so a batch beyond 2^31 points
    goes out in slices of 2^31 (xfxq2_smem.cu).  2^31 + 70 001 points, PID 21, a fifth of them below
    x_min: sampled against the oracle at both ends, across the slice boundary and at random."""
    torch = torch_cuda
    n = (1 << 31) + 70_001
    free, _ = torch.cuda.mem_get_info()
    if free < 3 * 8 * n + (8 << 30):
        pytest.skip("needs ~60 GB of free device memory")
    gen = torch.Generator(device="cuda").manual_seed(2009_06635)
    x = torch.empty(n, dtype=torch.float64, device="cuda")
    q2 = torch.empty(n, dtype=torch.float64, device="cuda")
    lx0, lq0, lq1 = np.log(float(grid2.x_knots[0])), np.log(grid2.q2_min), np.log(grid2.q2_max)
    step = 1 << 27
    for a in range(0, n, step):  # ln x uniform on [ln x_min - 5, 0]: about a fifth of the points below x_min
        b = min(n, a + step)
        x[a:b].uniform_(lx0 - 5.0, 0.0, generator=gen).exp_()
        q2[a:b].uniform_(lq0, lq1, generator=gen).exp_().clamp_(grid2.q2_min, grid2.q2_max)
    out = torch.full((1, n), -7.0, dtype=torch.float64, device="cuda")
    B.pdf_xfxq2(h2, [21], x, q2, out)
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    idx = np.unique(np.concatenate([np.arange(0, 2000), np.arange((1 << 31) - 3000, (1 << 31) + 3000), np.arange(n - 2000, n),
                                    rng.integers(0, n, 40_000)]))
    sel = torch.from_numpy(idx).cuda()
    xs, qs, got = x[sel].cpu().numpy(), q2[sel].cpu().numpy(), out[0, sel].cpu().numpy()
    ref, sc = ograph2.xfxq2([21], xs, qs, with_scale=True)
    st = check_parity(got[None, :], ref, sc, max_clause_frac=5e-3, what="2^31 + 70001 points")
    print("2^31 points", st, "below x_min in the sample:", float((xs < grid2.x_knots[0]).mean()))
    assert float((xs < grid2.x_knots[0]).mean()) > 0.1
    # nothing was left unwritten: no -7 anywhere (chunked, the array is 17 GB)
    for a in range(0, n, step):
        assert not bool((out[0, a:min(n, a + step)] == -7.0).any())


def test_host_threads_share_one_handle(torch_cuda, grid2, h2):
    """Four host threads (ctypes releases the GIL during a call), each on its own stream, launch small
    and large batches on ONE handle at the same time: the handle's only mutable host state is the
    round-robin slot counter (atomic) and the per-function attribute flags (atomic).  Every result
    equals the one the same call gives on its own."""
    import threading
    torch = torch_cuda
    pids = list(W.PIDS_11)
    work = []
    for k, n in enumerate((2_001, 40_003, 300_007, 5)):
        x, q2 = W.queries_extrapolation_mix(grid2, n, config=8000 + k)
        dx, dq = torch.from_numpy(x).cuda(), torch.from_numpy(q2).cuda()
        want = torch.empty((len(pids), n), dtype=torch.float64, device="cuda")
        B.pdf_xfxq2(h2, pids, dx, dq, want)
        work.append((dx, dq, want))
    torch.cuda.synchronize()
    errors = []

    def run(k):
        try:
            dx, dq, want = work[k]
            s = torch.cuda.Stream()
            for _ in range(40):
                out = torch.full_like(want, float("nan"))
                s.wait_stream(torch.cuda.current_stream())
                B.pdf_xfxq2(h2, pids, dx, dq, out, stream=s)
                s.synchronize()
                if not torch.equal(out.view(torch.int64), want.view(torch.int64)):
                    errors.append(k)
                    return
        except Exception as e:  # noqa: BLE001 -- reported below, from the main thread
            errors.append((k, repr(e)))

    threads = [threading.Thread(target=run, args=(k,)) for k in range(len(work))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
