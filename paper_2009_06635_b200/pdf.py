"""The user-facing object of the paper (Fig. 1): ``mkPDF()`` instantiates a ``PDF`` that
holds the grids of a set and exposes the interpolating methods -- two for the PDF (``xfxQ2``,
``xfxQ``) and two for alpha_s (``alphasQ2``, ``alphasQ``).  Everything here is marshalling: each
method allocates the output tensor and makes ONE call of the C-ABI library (binding.py); there is
no arithmetic of the method on this side and no fallback.  The paper's ``trace`` methods have no
counterpart: nothing is traced or compiled at run time.
"""
from __future__ import annotations

import os

import numpy as np

from . import binding as B


def _dev(t, device):
    import torch
    if isinstance(t, torch.Tensor):
        return t.to(device=f"cuda:{device}", dtype=torch.float64).contiguous()
    return torch.as_tensor(np.ascontiguousarray(t, dtype=np.float64), device=f"cuda:{device}")


class PDF:
    """A PDF set on one device: member tables on shared knots, plus (optionally) its alpha_s nodes."""

    def __init__(self, grid_handle, alphas_handle=None, pids=(), device: int = 0):
        self._g, self._a, self.device = grid_handle, alphas_handle, int(device)
        self.pids = tuple(int(p) for p in pids)
        self.n_members = B.pdf_set_members(grid_handle)

    # ---- the two interpolating methods of the PDF
    def xfxQ2(self, pids, x, q2, members=None, stream=None):
        """xf(x, Q^2): tensor [n_req, n] (member 0), or [n_members_requested, n_req, n] if ``members``
        is a (first, count) pair.  ``pids=None`` means every flavour of the set."""
        return self._xfx(pids, x, q2, members, stream, False)

    def xfxQ(self, pids, x, q, members=None, stream=None):
        """xf(x, Q) with Q in GeV; defined as xfxQ2 at Q*Q."""
        return self._xfx(pids, x, q, members, stream, True)

    def _xfx(self, pids, x, s, members, stream, s_is_q):
        import torch
        pids = list(self.pids) if pids is None else [int(p) for p in np.atleast_1d(pids)]
        xd, sd = _dev(x, self.device), _dev(s, self.device)
        n = xd.numel()
        if sd.numel() != n:
            raise ValueError("x and the scale array differ in length")
        with torch.cuda.device(self.device):
            if members is None:
                out = torch.empty((len(pids), n), dtype=torch.float64, device=xd.device)
                (B.pdf_xfxq if s_is_q else B.pdf_xfxq2)(self._g, pids, xd, sd, out, stream)
            else:
                m0, cnt = (int(v) for v in members)
                out = torch.empty((cnt, len(pids), n), dtype=torch.float64, device=xd.device)
                B.pdf_xfxq2_members(self._g, m0, cnt, pids, xd, sd, out, stream, q_is_q=s_is_q)
        return out

    # ---- the two interpolating methods of alpha_s
    def alphasQ2(self, q2, stream=None):
        return self._alphas(q2, stream, B.alphas_q2)

    def alphasQ(self, q, stream=None):
        return self._alphas(q, stream, B.alphas_q)

    def _alphas(self, s, stream, fn):
        import torch
        if self._a is None:
            raise RuntimeError("this PDF was made without alpha_s nodes")
        sd = _dev(s, self.device)
        with torch.cuda.device(self.device):
            out = torch.empty_like(sd)
            fn(self._a, sd, out, stream)
        return out

    def n_invalid(self) -> int:
        """Points so far that had no value (x > x_max, non-positive or NaN arguments)."""
        return B.pdf_grid_status(self._g)

    def close(self):
        if self._g is not None:
            B.pdf_grid_free(self._g)
            self._g = None
        if self._a is not None:
            B.alphas_grid_free(self._a)
            self._a = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def mkPDF(source, members=None, alphas=None, device: int = 0) -> PDF:
    """``source``: a directory in the LHAPDF6 text layout (``<dir>/<name>_NNNN.dat`` + ``<name>.info``),
    or a grid spec (workloads.PdfGridSpec), or a list of specs on the same knots (a set).
    ``members``: member numbers to load from a directory (default: all).  ``alphas``: an alpha_s spec
    for the spec forms."""
    if isinstance(source, (str, os.PathLike)):
        g, a, pids = B.load_lhapdf_set(os.fspath(source), members, device)
        return PDF(g, a, pids, device)
    specs = list(source) if isinstance(source, (list, tuple)) else [source]
    s0 = specs[0]
    g = B.pdf_set_load(s0.x_knots, s0.q_offsets, s0.q_knots, s0.pids, np.stack([s.values for s in specs]), device)
    a = B.load_alphas_spec(alphas, device) if alphas is not None else None
    return PDF(g, a, s0.pids, device)
