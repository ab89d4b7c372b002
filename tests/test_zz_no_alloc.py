"""alphas_q2_static: the entry point for callers that cannot allocate device memory.

Inside a TensorFlow-style process the framework's allocator has taken nearly the whole GPU, so the
cudaMalloc in alphas_grid_load can fail there; alphas_q2_static keeps its derived node table in a fixed
22 KB array that ships with the library instead (include/pdfb200.h).  All calls on a device share
that array, and it keeps the previous call's contents -- so the checks below always make at least two
calls in a row, with a different node list the second time, and compare each against the handle path
(alphas_grid_load + alphas_q2) within the tolerance every parity test of this suite uses.

This file sorts last on purpose (pytest -x stops at the first failure: a failure here hides nothing),
and it passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2009_06635_b200 import binding as B, workloads as W
from parity_util import check_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    torch.cuda.set_device(0)
    return torch


def _queries(spec, n, seed):
    """Q^2 over and beyond the node range, every node itself, and points without a value."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = spec.q_knots[0] ** 2, spec.q_knots[-1] ** 2
    q2 = np.exp(rng.uniform(np.log(lo) - 1.0, np.log(hi) + 1.0, n))
    nodes = spec.q_knots * spec.q_knots
    q2[: len(nodes)] = nodes
    q2[len(nodes): len(nodes) + 3] = (0.0, -1.0, np.nan)
    return q2


def _handle_path(torch, spec, dq):
    """The existing path: a handle (device allocation at load) and alphas_q2."""
    ha = B.load_alphas_spec(spec)
    out = torch.empty_like(dq)
    B.alphas_q2(ha, dq, out)
    torch.cuda.synchronize()
    B.alphas_grid_free(ha)
    return out.cpu().numpy()


def _long_list(n_nodes):
    """A node list of n_nodes nodes in 4 sub-grids, longer than the 192 nodes up to which alphas_q2
    switches to its table-logarithm kernel."""
    per = n_nodes // 4
    return W.make_alphas_grid(nq_per_sub=(per, per, per, n_nodes - 3 * per))


def test_static_scratch_matches_handle_path_on_two_calls_in_a_row(torch_cuda):
    torch = torch_cuda
    spec_a = W.make_alphas_grid()                                       # the suite's 4-sub-grid list
    spec_b = W.make_alphas_grid(jump=(1.0, 1.02, 1.0404, 1.061208))     # other values, steps at thresholds
    spec_c = _long_list(200)                                            # longer: rewrites more of the array
    n = 300_007                                                         # several grid-stride passes, ragged tail
    got, want = [], []
    # a -> c -> b -> a: a longer list after a shorter one, a shorter one on top of a longer one's
    # leftovers, and the first list again at the end
    for k, spec in enumerate((spec_a, spec_c, spec_b, spec_a)):
        dq = torch.from_numpy(_queries(spec, n, 77 + k)).cuda()
        out = torch.full_like(dq, 123.0)
        B.alphas_q2_static(spec.q_knots, spec.alphas, dq, out)          # back to back, no sync between calls
        got.append(out)
        want.append((spec, dq))
    torch.cuda.synchronize()
    for k, (out, (spec, dq)) in enumerate(zip(got, want)):
        ref = _handle_path(torch, spec, dq)
        res = out.cpu().numpy()
        assert np.array_equal(np.isnan(res), np.isnan(ref))
        check_parity(res, ref, what=f"alphas_q2_static call {k}")
    # the 200-node list is served by the general kernel on both sides: same bits
    assert np.array_equal(got[1].cpu().numpy(), _handle_path(torch, spec_c, want[1][1]), equal_nan=True)


def test_static_scratch_against_the_oracle(torch_cuda):
    import oracle
    torch = torch_cuda
    for k, spec in enumerate((W.make_alphas_grid(jump=(1.0, 1.02, 1.0404, 1.061208)), W.make_alphas_grid())):
        q2 = _queries(spec, 50_003, 5 + k)
        dq = torch.from_numpy(q2).cuda()
        out = torch.empty_like(dq)
        B.alphas_q2_static(spec.q_knots, spec.alphas, dq, out)
        torch.cuda.synchronize()
        check_parity(out.cpu().numpy(), oracle.OracleAlphas.from_spec(spec).q2(q2), what=f"alphas_q2_static oracle {k}")


def test_static_scratch_allocates_nothing_and_refuses_long_lists(torch_cuda):
    torch = torch_cuda
    spec = W.make_alphas_grid()
    dq = torch.from_numpy(_queries(spec, 10_001, 3)).cuda()
    out = torch.empty_like(dq)
    B.alphas_q2_static(spec.q_knots, spec.alphas, dq, out)              # set-up call of this device
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        B.alphas_q2_static(spec.q_knots, spec.alphas, dq, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                               # the device's free memory did not move
    # one node more than the array holds: a clear refusal, nothing launched, `out` untouched
    too_long = _long_list(B.PDFB_STATIC_MAX_KNOTS + 1)
    before = out.clone()
    launches = B.launch_count()
    with pytest.raises(B.PdfbError) as e:
        B.alphas_q2_static(too_long.q_knots, too_long.alphas, dq, out)
    assert e.value.code == B.PDFB_ESTATIC and "256" in str(e.value)
    assert B.launch_count() == launches
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.int64), before.view(torch.int64))     # (bit patterns: the batch holds NaN results)
    # exactly the maximum is served, and agrees with the handle path bit for bit (general kernel on both sides)
    full = _long_list(B.PDFB_STATIC_MAX_KNOTS)
    dq = torch.from_numpy(_queries(full, 20_011, 4)).cuda()
    out = torch.empty_like(dq)
    B.alphas_q2_static(full.q_knots, full.alphas, dq, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), _handle_path(torch, full, dq), equal_nan=True)
    # the node list is validated like alphas_grid_load's
    with pytest.raises(B.PdfbError) as e:
        B.alphas_q2_static([1.0, 2.0, 1.5], [0.3, 0.2, 0.25], dq, out)
    assert e.value.code == B.PDFB_EKNOTS
