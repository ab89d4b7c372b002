"""No-GPU checks of the boundary: the library loads, exports every symbol the header declares,
and validates arguments before touching CUDA."""
import ctypes
import re
import os

import numpy as np
import pytest

from paper_2009_06635_b200 import binding as B, build, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return B.lib()


def test_exports_every_declared_symbol(L):
    hdr = open(os.path.join(ROOT, "include", "pdfb200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(pdf_\w+|alphas_\w+|pdfb_\w+)\s*\(", hdr))
    assert {"pdf_grid_load", "pdf_xfxq2", "alphas_grid_load", "alphas_q2"} <= names
    for n in names:
        assert hasattr(L, n), n
    assert set(B.EXPORTS) <= names
    assert "pdfb_probe" not in names and not hasattr(L, "pdfb_probe")  # the bench's machine probes are not in the product library


def test_probe_library_exports_its_header(L):
    """include/pdfb200_probe.h is served by libpdfb200_probe.so, a library of its own."""
    import ctypes
    hdr = open(os.path.join(ROOT, "include", "pdfb200_probe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(pdfb_\w+)\s*\(", hdr))
    assert names == {"pdfb_probe"}
    P = ctypes.CDLL(build.PROBE_LIB)
    for n in names:
        assert hasattr(P, n), n


def test_strerror_and_codes(L):
    assert B.strerror(0) == "ok"
    for c in (-1, -2, -3, -4, -5, -99):
        assert len(B.strerror(c)) > 3


def test_load_validates_before_cuda(L):
    g = W.grid_config1()
    bad_x = g.x_knots.copy(); bad_x[3] = bad_x[2]
    with pytest.raises(B.PdfbError) as e:
        B.pdf_grid_load(bad_x, g.q_offsets, g.q_knots, g.pids, g.values)
    assert e.value.code == -2
    g2 = W.grid_nnpdf_shaped()
    bad_q = g2.q_knots.copy(); bad_q[7] *= 1.0001  # sub-grid 1 no longer starts at the threshold
    with pytest.raises(B.PdfbError) as e:
        B.pdf_grid_load(g2.x_knots, g2.q_offsets, bad_q, g2.pids, g2.values)
    assert e.value.code == -2
    with pytest.raises(B.PdfbError) as e:  # a sub-grid with one knot
        B.pdf_grid_load(g.x_knots, np.array([0, 1, 15], np.int32), g.q_knots, g.pids, g.values)
    assert e.value.code == -2
    bad_v = g.values.copy(); bad_v[17] = np.inf       # table values must be finite
    with pytest.raises(B.PdfbError) as e:
        B.pdf_grid_load(g.x_knots, g.q_offsets, g.q_knots, g.pids, bad_v)
    assert e.value.code == -1
    with pytest.raises(B.PdfbError) as e:             # member count out of range
        B.pdf_set_load(g.x_knots, g.q_offsets, g.q_knots, g.pids, np.zeros((0, g.values.size)))
    assert e.value.code == -5
    with pytest.raises(B.PdfbError) as e:
        B.alphas_grid_load([1.0, 2.0, 1.5], [0.3, 0.2, 0.25])
    assert e.value.code == -2
    with pytest.raises(B.PdfbError) as e:
        B.alphas_grid_load([1.0, 2.0, 2.0], [0.3, 0.2, 0.25])  # upper sub-grid has one node
    assert e.value.code == -2


def test_no_device_is_a_loud_error(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    g = W.grid_config1()
    with pytest.raises(B.PdfbError) as e:
        B.load_pdf_spec(g)
    assert e.value.code == -4  # PDFB_ECUDA: there is no CPU fallback


def test_null_handles_rejected(L):
    rc = L.pdf_xfxq2(None, 1, (ctypes.c_int * 1)(21), 0, None, None, None, None)
    assert rc == -1
    rc = L.alphas_q2(None, 0, None, None, None)
    assert rc == -1


def test_alphas_q2_static_validates_before_cuda(L):
    """The no-allocation entry point checks its node list on the host, before any CUDA call: a list
    longer than its fixed scratch array holds is refused with a code of its own."""
    qk = np.geomspace(1.0, 1e4, B.PDFB_STATIC_MAX_KNOTS + 1)
    al = np.linspace(0.3, 0.1, len(qk))
    dp = ctypes.POINTER(ctypes.c_double)
    rc = L.alphas_q2_static(len(qk), qk.ctypes.data_as(dp), al.ctypes.data_as(dp), 0, None, None, None)
    assert rc == B.PDFB_ESTATIC and "256" in B.strerror(rc)
    qk, al = qk[:-1].copy(), al[:-1].copy()
    assert L.alphas_q2_static(len(qk), qk.ctypes.data_as(dp), al.ctypes.data_as(dp), 0, None, None, None) == 0   # n = 0: nothing to do
    assert L.alphas_q2_static(len(qk), qk.ctypes.data_as(dp), al.ctypes.data_as(dp), 5, None, None, None) == B.PDFB_EINVAL
    assert L.alphas_q2_static(1, qk.ctypes.data_as(dp), al.ctypes.data_as(dp), 0, None, None, None) == B.PDFB_EINVAL
    qk[7] = qk[6] * 0.5
    assert L.alphas_q2_static(len(qk), qk.ctypes.data_as(dp), al.ctypes.data_as(dp), 0, None, None, None) == B.PDFB_EKNOTS
    hdr = open(os.path.join(ROOT, "include", "pdfb200.h")).read()
    assert f"#define PDFB_STATIC_MAX_KNOTS {B.PDFB_STATIC_MAX_KNOTS}" in hdr
