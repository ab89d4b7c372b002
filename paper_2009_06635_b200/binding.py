"""Thin ctypes binding of include/pdfb200.h -- argument marshalling only.

Same names as the C-ABI.  Host arrays are numpy; device arrays are torch CUDA tensors (torch
supplies device memory and streams, nothing else).  There is no fallback: if libpdfb200.so is
missing or does not load, ``lib()`` raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpdfb200.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_vp = ctypes.c_void_p
_ll = ctypes.c_longlong

EXPORTS = ("pdf_grid_load", "pdf_set_load", "pdf_set_members", "pdf_xfxq2_members", "pdf_xfxq_members", "pdf_xfxq2", "pdf_xfxq", "alphas_q", "pdf_xfxq2_host", "pdf_grid_status", "pdf_grid_free",
           "alphas_grid_load", "alphas_q2", "alphas_q2_host", "alphas_grid_free", "pdfb_strerror",
           "pdfb_launch_count", "pdf_lumi_events", "pdf_xfxq2_pm", "pdf_xfxq2_f32", "pdf_grid_load_xs", "pdfb_lhagrid_dims_xs", "pdfb_lhagrid_get_xs", "pdfb_lhagrid_read", "pdfb_lhagrid_dims", "pdfb_lhagrid_get",
           "pdfb_lhagrid_free", "pdfb_lhapdf_info_alphas", "pdfb_lhapdf_info_members", "alphas_q2_static")


PDFB_EINVAL, PDFB_EKNOTS, PDFB_EPID, PDFB_ECUDA, PDFB_ELIMIT, PDFB_EIO, PDFB_EFORMAT, PDFB_EXKNOTS = -1, -2, -3, -4, -5, -6, -7, -8
PDFB_ESTATIC = -9
PDFB_STATIC_MAX_KNOTS = 256


class PdfbError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} (code {code})")


def lib():
    """Load libpdfb200.so (built in-tree by ``paper_2009_06635_b200.build``); fail loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2009_06635_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        L.pdf_grid_load.restype = ctypes.c_int
        L.pdf_grid_load.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _ip, _dp, ctypes.c_int, _ip, _dp,
                                    ctypes.c_int, ctypes.POINTER(_vp)]
        L.pdf_set_load.restype = ctypes.c_int
        L.pdf_set_load.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _dp, _ip, _dp, ctypes.c_int, _ip, _dp,
                                   ctypes.c_int, ctypes.POINTER(_vp)]
        L.pdf_set_members.restype = ctypes.c_int
        L.pdf_set_members.argtypes = [_vp]
        L.pdf_xfxq2_members.restype = ctypes.c_int
        L.pdf_xfxq2_members.argtypes = [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _ip, _ll, _vp, _vp, _vp, _vp]
        L.pdf_xfxq_members.restype = ctypes.c_int
        L.pdf_xfxq_members.argtypes = [_vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, _ip, _ll, _vp, _vp, _vp, _vp]
        for fn in (L.pdf_xfxq2_pm, L.pdf_xfxq2_f32):
            fn.restype = ctypes.c_int
            fn.argtypes = [_vp, ctypes.c_int, _ip, _ll, _vp, _vp, _vp, _vp]
        L.pdf_lumi_events.restype = ctypes.c_int
        L.pdf_lumi_events.argtypes = [_vp, _vp, ctypes.c_int, _ip, _ip, _dp, _ll, _vp, _vp, _vp, _vp, _vp, ctypes.c_int, _vp]
        L.pdf_xfxq2.restype = ctypes.c_int
        L.pdf_xfxq2.argtypes = [_vp, ctypes.c_int, _ip, _ll, _vp, _vp, _vp, _vp]
        L.pdf_xfxq.restype = ctypes.c_int
        L.pdf_xfxq.argtypes = [_vp, ctypes.c_int, _ip, _ll, _vp, _vp, _vp, _vp]
        L.alphas_q.restype = ctypes.c_int
        L.alphas_q.argtypes = [_vp, _ll, _vp, _vp, _vp]
        L.pdf_xfxq2_host.restype = ctypes.c_int
        L.pdf_xfxq2_host.argtypes = [_vp, ctypes.c_int, _ip, _ll, _vp, _vp, _vp]
        L.pdf_grid_status.restype = ctypes.c_int
        L.pdf_grid_status.argtypes = [_vp, ctypes.POINTER(_ll)]
        L.pdf_grid_free.restype = None
        L.pdf_grid_free.argtypes = [_vp]
        L.pdf_grid_setup_ms.restype = ctypes.c_double
        L.pdf_grid_setup_ms.argtypes = [_vp]
        L.pdf_grid_uses_smem_path.restype = ctypes.c_int
        L.pdf_grid_uses_smem_path.argtypes = [_vp]
        L.alphas_grid_load.restype = ctypes.c_int
        L.alphas_grid_load.argtypes = [ctypes.c_int, _dp, _dp, ctypes.c_int, ctypes.POINTER(_vp)]
        L.alphas_q2.restype = ctypes.c_int
        L.alphas_q2.argtypes = [_vp, _ll, _vp, _vp, _vp]
        L.alphas_q2_host.restype = ctypes.c_int
        L.alphas_q2_host.argtypes = [_vp, _ll, _vp, _vp]
        L.alphas_q2_static.restype = ctypes.c_int
        L.alphas_q2_static.argtypes = [ctypes.c_int, _dp, _dp, _ll, _vp, _vp, _vp]
        L.alphas_grid_free.restype = None
        L.alphas_grid_free.argtypes = [_vp]
        L.pdfb_strerror.restype = ctypes.c_char_p
        L.pdfb_strerror.argtypes = [ctypes.c_int]
        L.pdfb_launch_count.restype = _ll
        L.pdfb_lhagrid_read.restype = ctypes.c_int
        L.pdfb_lhagrid_read.argtypes = [ctypes.c_char_p, ctypes.POINTER(_vp)]
        L.pdfb_lhagrid_dims.restype = ctypes.c_int
        L.pdfb_lhagrid_dims.argtypes = [_vp, _ip, _ip, _ip, _ip]
        L.pdfb_lhagrid_get.restype = ctypes.c_int
        L.pdfb_lhagrid_get.argtypes = [_vp, _dp, _ip, _dp, _ip, _dp]
        L.pdfb_lhagrid_free.restype = None
        L.pdfb_lhagrid_free.argtypes = [_vp]
        L.pdfb_lhapdf_info_alphas.restype = ctypes.c_int
        L.pdfb_lhapdf_info_alphas.argtypes = [ctypes.c_char_p, ctypes.c_int, _dp, _dp, _ip]
        L.pdfb_lhapdf_info_members.restype = ctypes.c_int
        L.pdfb_lhapdf_info_members.argtypes = [ctypes.c_char_p, _ip]
        L.pdfb_debug_ln.restype = ctypes.c_int
        L.pdfb_debug_ln.argtypes = [_vp, _vp, _ll, _vp]
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().pdfb_strerror(int(code)).decode()


def launch_count() -> int:
    return int(lib().pdfb_launch_count())


PROBE_FP64, PROBE_LDS = 1, 2


_probe_lib = None


def probe(which: int, device: int = 0) -> float:
    """Machine probe (include/pdfb200_probe.h, libpdfb200_probe.so -- a bench utility, not part of the
    product library): FP64 FMA/s or shared-memory bytes/s."""
    global _probe_lib
    if _probe_lib is None:
        path = os.path.join(_HERE, "libpdfb200_probe.so")
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: build it with `python -m paper_2009_06635_b200.build`")
        _probe_lib = ctypes.CDLL(path)
        _probe_lib.pdfb_probe.restype = ctypes.c_int
        _probe_lib.pdfb_probe.argtypes = [ctypes.c_int, ctypes.c_int, _dp]
    r = ctypes.c_double(0.0)
    _check(_probe_lib.pdfb_probe(int(which), int(device), ctypes.byref(r)), "pdfb_probe")
    return r.value


def debug_ln(x, out, stream=None):
    n = int(x.numel())
    _check(lib().pdfb_debug_ln(_dev_ptr(x, n, "x"), _dev_ptr(out, n, "out"), n, _stream_ptr(stream)), "pdfb_debug_ln")


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(np.atleast_1d(a), dtype=np.int32)


def _check(rc: int, where: str):
    if rc != 0:
        raise PdfbError(rc, where)


def _dev_ptr(t, n, name, dtype="float64"):
    """Pointer of a contiguous CUDA tensor of the given dtype with at least n elements."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == getattr(torch, dtype) and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous {dtype} CUDA tensor")
    if t.numel() < n:
        raise ValueError(f"{name} has {t.numel()} elements, need {n}")
    return ctypes.c_void_p(t.data_ptr())


def _host_ptr(a, n, name):
    """Pointer of host memory: numpy float64 array or CPU (possibly pinned) torch tensor."""
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags.c_contiguous or a.size < n:
            raise TypeError(f"{name} must be a C-contiguous float64 array with >= {n} elements")
        return ctypes.c_void_p(a.ctypes.data)
    import torch
    if isinstance(a, torch.Tensor) and not a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() \
            and a.numel() >= n:
        return ctypes.c_void_p(a.data_ptr())
    raise TypeError(f"{name} must be host float64 memory with >= {n} elements")


def _stream_ptr(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


# ------------------------------------------------------------------ the C-ABI calls
def pdf_grid_load(x_knots, q_offsets, q_knots, pids, values, device: int = 0):
    """-> opaque handle (int).  Arguments as in pdfb200.h; host numpy arrays."""
    x_knots, q_knots, values = _f64(x_knots), _f64(q_knots), _f64(values)
    q_offsets, pids = _i32(q_offsets), _i32(pids)
    h = _vp()
    rc = lib().pdf_grid_load(len(q_offsets) - 1, len(x_knots), x_knots.ctypes.data_as(_dp),
                             q_offsets.ctypes.data_as(_ip), q_knots.ctypes.data_as(_dp), len(pids),
                             pids.ctypes.data_as(_ip), values.ctypes.data_as(_dp), int(device),
                             ctypes.byref(h))
    _check(rc, "pdf_grid_load")
    return h.value


def pdf_grid_load_xs(x_offsets, x_knots, q_offsets, q_knots, pids, values, device: int = 0):
    """A member whose sub-grids have their own x-knot arrays (x_knots = the arrays one after the other,
    x_offsets delimits them; values [s][ix_s][iq_s][ipid]) -> opaque handle."""
    x_knots, q_knots, values = _f64(x_knots), _f64(q_knots), _f64(values)
    x_offsets, q_offsets, pids = _i32(x_offsets), _i32(q_offsets), _i32(pids)
    h = _vp()
    L = lib()
    L.pdf_grid_load_xs.restype = ctypes.c_int
    L.pdf_grid_load_xs.argtypes = [ctypes.c_int, _ip, _dp, _ip, _dp, ctypes.c_int, _ip, _dp, ctypes.c_int, ctypes.POINTER(_vp)]
    rc = L.pdf_grid_load_xs(len(q_offsets) - 1, x_offsets.ctypes.data_as(_ip), x_knots.ctypes.data_as(_dp),
                            q_offsets.ctypes.data_as(_ip), q_knots.ctypes.data_as(_dp), len(pids),
                            pids.ctypes.data_as(_ip), values.ctypes.data_as(_dp), int(device), ctypes.byref(h))
    _check(rc, "pdf_grid_load_xs")
    return h.value


def pdf_set_load(x_knots, q_offsets, q_knots, pids, values, device: int = 0):
    """-> handle of a PDF set; values[member] = one member's table in LHAPDF grid-file order."""
    x_knots, q_knots = _f64(x_knots), _f64(q_knots)
    q_offsets, pids = _i32(q_offsets), _i32(pids)
    values = _f64(values)
    if values.ndim != 2:
        raise ValueError("values must be [n_members, table size]")
    h = _vp()
    rc = lib().pdf_set_load(values.shape[0], len(q_offsets) - 1, len(x_knots), x_knots.ctypes.data_as(_dp),
                            q_offsets.ctypes.data_as(_ip), q_knots.ctypes.data_as(_dp), len(pids),
                            pids.ctypes.data_as(_ip), values.ctypes.data_as(_dp), int(device), ctypes.byref(h))
    _check(rc, "pdf_set_load")
    return h.value


def pdf_set_members(g) -> int:
    return int(lib().pdf_set_members(_vp(g)))


def pdf_xfxq2_members(g, member0, n_mem, pids, x, q2, out, stream=None, n=None, q_is_q=False):
    """Enqueue members member0..member0+n_mem-1 on the same points -> out[n_mem, n_req, n]."""
    pids = _i32(pids)
    n = int(x.numel() if n is None else n)
    rc = (lib().pdf_xfxq_members if q_is_q else lib().pdf_xfxq2_members)(_vp(g), int(member0), int(n_mem), len(pids), pids.ctypes.data_as(_ip), n,
                                 _dev_ptr(x, n, "x"), _dev_ptr(q2, n, "q2"),
                                 _dev_ptr(out, int(n_mem) * len(pids) * n, "out"), _stream_ptr(stream))
    _check(rc, "pdf_xfxq2_members")


def pdf_xfxq2(g, pids, x, q2, out, stream=None, n=None):
    """Enqueue xf(x,Q^2) for device tensors x, q2 -> out[n_req, n] on `stream` (torch current)."""
    pids = _i32(pids)
    n = int(x.numel() if n is None else n)
    rc = lib().pdf_xfxq2(_vp(g), len(pids), pids.ctypes.data_as(_ip), n, _dev_ptr(x, n, "x"),
                         _dev_ptr(q2, n, "q2"), _dev_ptr(out, len(pids) * n, "out"), _stream_ptr(stream))
    _check(rc, "pdf_xfxq2")


def pdf_lumi_events(g, terms, x1, x2, q2, lumi, alphas=None, alphas_out=None, divide_by_x=False, stream=None, n=None):
    """Enqueue the fused parton luminosity sum_t c_t xf_a(x1,Q2) xf_b(x2,Q2) for device tensors -> lumi[n]
    (and alpha_s(Q2) -> alphas_out[n] if an alpha_s handle is given).  terms: iterable of (pid_a, pid_b, c)."""
    terms = list(terms)
    pa, pb = _i32([t[0] for t in terms]), _i32([t[1] for t in terms])
    cc = _f64([t[2] for t in terms])
    n = int(x1.numel() if n is None else n)
    rc = lib().pdf_lumi_events(_vp(g), _vp(alphas) if alphas is not None else None, len(terms), pa.ctypes.data_as(_ip),
                               pb.ctypes.data_as(_ip), cc.ctypes.data_as(_dp), n, _dev_ptr(x1, n, "x1"), _dev_ptr(x2, n, "x2"),
                               _dev_ptr(q2, n, "q2"), _dev_ptr(lumi, n, "lumi"),
                               _dev_ptr(alphas_out, n, "alphas_out") if alphas_out is not None else None,
                               1 if divide_by_x else 0, _stream_ptr(stream))
    _check(rc, "pdf_lumi_events")


def pdf_xfxq2_pm(g, pids, x, q2, out, stream=None, n=None):
    """pdf_xfxq2 with point-major output: out[n, n_req] (fp64)."""
    pids = _i32(pids)
    n = int(x.numel() if n is None else n)
    rc = lib().pdf_xfxq2_pm(_vp(g), len(pids), pids.ctypes.data_as(_ip), n, _dev_ptr(x, n, "x"),
                            _dev_ptr(q2, n, "q2"), _dev_ptr(out, len(pids) * n, "out"), _stream_ptr(stream))
    _check(rc, "pdf_xfxq2_pm")


def pdf_xfxq2_f32(g, pids, x, q2, out, stream=None, n=None):
    """pdf_xfxq2 with fp32 output (fp64 arithmetic, one rounding at the store): out[n_req, n] float32."""
    pids = _i32(pids)
    n = int(x.numel() if n is None else n)
    rc = lib().pdf_xfxq2_f32(_vp(g), len(pids), pids.ctypes.data_as(_ip), n, _dev_ptr(x, n, "x"),
                             _dev_ptr(q2, n, "q2"), _dev_ptr(out, len(pids) * n, "out", dtype="float32"), _stream_ptr(stream))
    _check(rc, "pdf_xfxq2_f32")


def pdf_xfxq(g, pids, x, q, out, stream=None, n=None):
    """Enqueue xf(x,Q), Q in GeV, for device tensors x, q -> out[n_req, n] on `stream`."""
    pids = _i32(pids)
    n = int(x.numel() if n is None else n)
    rc = lib().pdf_xfxq(_vp(g), len(pids), pids.ctypes.data_as(_ip), n, _dev_ptr(x, n, "x"),
                        _dev_ptr(q, n, "q"), _dev_ptr(out, len(pids) * n, "out"), _stream_ptr(stream))
    _check(rc, "pdf_xfxq")


def pdf_xfxq2_host(g, pids, x, q2, out):
    """Synchronous evaluation for HOST buffers (numpy or pinned torch CPU tensors)."""
    pids = _i32(pids)
    n = int(x.size if isinstance(x, np.ndarray) else x.numel())
    rc = lib().pdf_xfxq2_host(_vp(g), len(pids), pids.ctypes.data_as(_ip), n, _host_ptr(x, n, "x"),
                              _host_ptr(q2, n, "q2"), _host_ptr(out, len(pids) * n, "out"))
    _check(rc, "pdf_xfxq2_host")


def pdf_grid_status(g) -> int:
    c = _ll(0)
    _check(lib().pdf_grid_status(_vp(g), ctypes.byref(c)), "pdf_grid_status")
    return int(c.value)


def pdf_grid_setup_ms(g) -> float:
    return float(lib().pdf_grid_setup_ms(_vp(g)))


def pdf_grid_uses_smem_path(g) -> bool:
    return bool(lib().pdf_grid_uses_smem_path(_vp(g)))


def pdf_grid_free(g):
    lib().pdf_grid_free(_vp(g))


def alphas_grid_load(q_knots, alphas, device: int = 0):
    q_knots, alphas = _f64(q_knots), _f64(alphas)
    if q_knots.shape != alphas.shape:
        raise ValueError("q_knots and alphas differ in length")
    h = _vp()
    rc = lib().alphas_grid_load(len(q_knots), q_knots.ctypes.data_as(_dp), alphas.ctypes.data_as(_dp),
                                int(device), ctypes.byref(h))
    _check(rc, "alphas_grid_load")
    return h.value


def alphas_q2(a, q2, out, stream=None, n=None):
    n = int(q2.numel() if n is None else n)
    rc = lib().alphas_q2(_vp(a), n, _dev_ptr(q2, n, "q2"), _dev_ptr(out, n, "out"), _stream_ptr(stream))
    _check(rc, "alphas_q2")


def alphas_q(a, q, out, stream=None, n=None):
    n = int(q.numel() if n is None else n)
    rc = lib().alphas_q(_vp(a), n, _dev_ptr(q, n, "q"), _dev_ptr(out, n, "out"), _stream_ptr(stream))
    _check(rc, "alphas_q")


def alphas_q2_host(a, q2, out):
    n = int(q2.size if isinstance(q2, np.ndarray) else q2.numel())
    rc = lib().alphas_q2_host(_vp(a), n, _host_ptr(q2, n, "q2"), _host_ptr(out, n, "out"))
    _check(rc, "alphas_q2_host")


def alphas_q2_static(q_knots, alphas, q2, out, stream=None, n=None):
    """alpha_s(Q^2) without a handle and without any device allocation (include/pdfb200.h): for use
    inside a process whose framework owns the GPU's memory pool, where the library's own cudaMalloc
    would fail.  q_knots / alphas: host node list of at most PDFB_STATIC_MAX_KNOTS nodes; q2 / out:
    torch CUDA tensors on the current device.  Calls that overlap on the GPU race on the shared table."""
    q_knots, alphas = _f64(q_knots), _f64(alphas)
    if q_knots.shape != alphas.shape:
        raise ValueError("q_knots and alphas differ in length")
    n = int(q2.numel() if n is None else n)
    rc = lib().alphas_q2_static(len(q_knots), q_knots.ctypes.data_as(_dp), alphas.ctypes.data_as(_dp), n,
                                _dev_ptr(q2, n, "q2"), _dev_ptr(out, n, "out"), _stream_ptr(stream))
    _check(rc, "alphas_q2_static")


def alphas_grid_free(a):
    lib().alphas_grid_free(_vp(a))


# ------------------------------------------------------------------ LHAPDF text layout (host only)
def lhagrid_read(path: str):
    """Parse one member file -> (x_knots, q_offsets, q_knots, pids, values), pdf_grid_load's arguments."""
    h = _vp()
    _check(lib().pdfb_lhagrid_read(os.fsencode(path), ctypes.byref(h)), f"pdfb_lhagrid_read({path})")
    try:
        d = [ctypes.c_int(0) for _ in range(4)]
        _check(lib().pdfb_lhagrid_dims(h, *[ctypes.byref(v) for v in d]), "pdfb_lhagrid_dims")
        n_sub, nx, nq_tot, n_pid = (int(v.value) for v in d)
        x, q = np.empty(nx), np.empty(nq_tot)
        off, pids = np.empty(n_sub + 1, np.int32), np.empty(n_pid, np.int32)
        vals = np.empty(nx * nq_tot * n_pid)
        _check(lib().pdfb_lhagrid_get(h, x.ctypes.data_as(_dp), off.ctypes.data_as(_ip), q.ctypes.data_as(_dp),
                                      pids.ctypes.data_as(_ip), vals.ctypes.data_as(_dp)), "pdfb_lhagrid_get")
    finally:
        lib().pdfb_lhagrid_free(h)
    return x, off, q, pids, vals


def lhagrid_read_xs(path: str):
    """Parse one member file whose sub-grids may carry their own x-knot arrays ->
    (x_offsets, x_knots, q_offsets, q_knots, pids, values, shared_x): pdf_grid_load_xs's arguments."""
    h = _vp()
    L = lib()
    L.pdfb_lhagrid_dims_xs.restype = ctypes.c_int
    L.pdfb_lhagrid_dims_xs.argtypes = [_vp] + [ctypes.POINTER(ctypes.c_int)] * 4 + [ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(ctypes.c_int)]
    L.pdfb_lhagrid_get_xs.restype = ctypes.c_int
    L.pdfb_lhagrid_get_xs.argtypes = [_vp, _ip, _dp, _ip, _dp, _ip, _dp]
    _check(L.pdfb_lhagrid_read(os.fsencode(path), ctypes.byref(h)), f"pdfb_lhagrid_read({path})")
    try:
        d = [ctypes.c_int(0) for _ in range(4)]
        nv, sh = ctypes.c_longlong(0), ctypes.c_int(0)
        _check(L.pdfb_lhagrid_dims_xs(h, *[ctypes.byref(v) for v in d], ctypes.byref(nv), ctypes.byref(sh)), "pdfb_lhagrid_dims_xs")
        n_sub, nxt, nq_tot, n_pid = (int(v.value) for v in d)
        x, q = np.empty(nxt), np.empty(nq_tot)
        xoff, off, pids = np.empty(n_sub + 1, np.int32), np.empty(n_sub + 1, np.int32), np.empty(n_pid, np.int32)
        vals = np.empty(int(nv.value))
        _check(L.pdfb_lhagrid_get_xs(h, xoff.ctypes.data_as(_ip), x.ctypes.data_as(_dp), off.ctypes.data_as(_ip),
                                     q.ctypes.data_as(_dp), pids.ctypes.data_as(_ip), vals.ctypes.data_as(_dp)), "pdfb_lhagrid_get_xs")
    finally:
        L.pdfb_lhagrid_free(h)
    return xoff, x, off, q, pids, vals, bool(sh.value)


def lhapdf_info_alphas(info_path: str):
    """-> (q_knots, alphas) of a set's metadata file."""
    n = ctypes.c_int(0)
    _check(lib().pdfb_lhapdf_info_alphas(os.fsencode(info_path), 0, None, None, ctypes.byref(n)), "pdfb_lhapdf_info_alphas")
    q, a = np.empty(n.value), np.empty(n.value)
    _check(lib().pdfb_lhapdf_info_alphas(os.fsencode(info_path), n.value, q.ctypes.data_as(_dp), a.ctypes.data_as(_dp),
                                         ctypes.byref(n)), "pdfb_lhapdf_info_alphas")
    return q, a


def lhapdf_info_members(info_path: str) -> int:
    n = ctypes.c_int(0)
    _check(lib().pdfb_lhapdf_info_members(os.fsencode(info_path), ctypes.byref(n)), "pdfb_lhapdf_info_members")
    return int(n.value)


def load_lhapdf_set(set_dir: str, members=None, device: int = 0):
    """Load <set_dir>/<name>_NNNN.dat (name = directory name) as a PDF set and the alpha_s nodes of
    <name>.info -> (pdf handle, alphas handle, PIDs).  members: iterable of member numbers (default all)."""
    name = os.path.basename(os.path.normpath(set_dir))
    info = os.path.join(set_dir, name + ".info")
    if members is None:
        members = range(lhapdf_info_members(info))
    first, tables = None, []
    members = list(members)
    xs = lhagrid_read_xs(os.path.join(set_dir, f"{name}_{int(members[0]):04d}.dat"))
    if not xs[6]:  # sub-grids with their own x-knot arrays: one member, read-only-cache kernel
        if len(members) != 1:
            raise PdfbError(PDFB_EXKNOTS, f"{name}: sets whose sub-grids carry their own x-knot arrays load one member at a time")
        hp = pdf_grid_load_xs(xs[0], xs[1], xs[2], xs[3], xs[4], xs[5], device)
        qa, aa = lhapdf_info_alphas(info)
        return hp, alphas_grid_load(qa, aa, device), xs[4]
    for m in members:
        x, off, q, pids, vals = lhagrid_read(os.path.join(set_dir, f"{name}_{int(m):04d}.dat"))
        if first is None:
            first = (x, off, q, pids)
        elif not (np.array_equal(x, first[0]) and np.array_equal(off, first[1]) and np.array_equal(q, first[2])
                  and np.array_equal(pids, first[3])):
            raise PdfbError(-2, f"member {m} of {name} is on different knots")
        tables.append(vals)
    hp = pdf_set_load(first[0], first[1], first[2], first[3], np.stack(tables), device)
    qa, aa = lhapdf_info_alphas(info)
    return hp, alphas_grid_load(qa, aa, device), first[3]


# ------------------------------------------------------------------ spec conveniences
def load_pdf_spec(spec, device: int = 0):
    if getattr(spec, "x_offsets", None) is not None:
        return pdf_grid_load_xs(spec.x_offsets, spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, spec.values, device)
    return pdf_grid_load(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, spec.values, device)


def load_alphas_spec(spec, device: int = 0):
    return alphas_grid_load(spec.q_knots, spec.alphas, device)
