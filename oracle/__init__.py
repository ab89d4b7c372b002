"""CPU oracle -- TEST INFRASTRUCTURE, not the product.

Thin ctypes access to ``oracle/pdf_oracle.c`` (plain scalar C, fp64).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2009_06635_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdf_oracle.c")
_LIB = os.path.join(_HERE, "libpdforacle.so")
_lib = None

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
               "-o", _LIB, _SRC, "-lquadmath", "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_pdf_grid_create.restype = ctypes.c_void_p
        lib.oracle_pdf_grid_create.argtypes = [ctypes.c_int, ctypes.c_int, _dp, _ip, _dp,
                                               ctypes.c_int, _ip, _dp]
        lib.oracle_pdf_grid_create_xs.restype = ctypes.c_void_p
        lib.oracle_pdf_grid_create_xs.argtypes = [ctypes.c_int, ctypes.c_int, _ip, _dp, _ip, _dp,
                                                  ctypes.c_int, _ip, _dp]
        lib.oracle_pdf_grid_free.argtypes = [ctypes.c_void_p]
        lib.oracle_pdf_grid_invalid.restype = ctypes.c_long
        lib.oracle_pdf_grid_invalid.argtypes = [ctypes.c_void_p]
        lib.oracle_pdf_xfxq2.restype = ctypes.c_int
        lib.oracle_pdf_xfxq2.argtypes = [ctypes.c_void_p, ctypes.c_int, _ip, ctypes.c_long,
                                         _dp, _dp, _dp, _dp]
        lib.oracle_alphas_create.restype = ctypes.c_void_p
        lib.oracle_alphas_create.argtypes = [ctypes.c_int, _dp, _dp]
        lib.oracle_alphas_free.argtypes = [ctypes.c_void_p]
        lib.oracle_alphas_q2.restype = ctypes.c_int
        lib.oracle_alphas_q2.argtypes = [ctypes.c_void_p, ctypes.c_long, _dp, _dp]
        lib.oracle_ln.restype = ctypes.c_double
        lib.oracle_ln.argtypes = [ctypes.c_double]
        lib.oracle_threads.restype = ctypes.c_int
        lib.oracle_set_threads.argtypes = [ctypes.c_int]
        _lib = lib
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def threads() -> int:
    return int(_load().oracle_threads())


def set_threads(n: int) -> None:
    _load().oracle_set_threads(int(n))


def ln(a: float) -> float:
    return float(_load().oracle_ln(float(a)))


class OraclePdfGrid:
    """Oracle-side grid (arguments as in the C-ABI's pdf_grid_load)."""

    def __init__(self, x_knots, q_offsets, q_knots, pids, values, x_offsets=None):
        """x_offsets (n_sub + 1 entries into x_knots): every sub-grid has its own x-knot array and the
        values are [s][ix_s][iq_s][ipid]; None: one x-knot array shared by all sub-grids."""
        lib = _load()
        x_knots, q_knots, values = _f64(x_knots), _f64(q_knots), _f64(values)
        q_offsets, pids = _i32(q_offsets), _i32(pids)
        if x_offsets is None:
            self._h = lib.oracle_pdf_grid_create(
                len(q_offsets) - 1, len(x_knots), x_knots.ctypes.data_as(_dp),
                q_offsets.ctypes.data_as(_ip), q_knots.ctypes.data_as(_dp), len(pids),
                pids.ctypes.data_as(_ip), values.ctypes.data_as(_dp))
        else:
            x_offsets = _i32(x_offsets)
            self._h = lib.oracle_pdf_grid_create_xs(
                len(q_offsets) - 1, 0, x_offsets.ctypes.data_as(_ip), x_knots.ctypes.data_as(_dp),
                q_offsets.ctypes.data_as(_ip), q_knots.ctypes.data_as(_dp), len(pids),
                pids.ctypes.data_as(_ip), values.ctypes.data_as(_dp))

    @classmethod
    def from_spec(cls, spec):
        return cls(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, spec.values,
                   x_offsets=getattr(spec, "x_offsets", None))

    def xfxq2(self, pids, x, q2, with_scale: bool = False):
        """-> out[n_req, n] (flavour-major); with_scale also returns the conditioning scale."""
        lib = _load()
        pids, x, q2 = _i32(np.atleast_1d(pids)), _f64(np.atleast_1d(x)), _f64(np.atleast_1d(q2))
        assert x.shape == q2.shape and x.ndim == 1
        n = x.shape[0]
        out = np.empty((len(pids), n), dtype=np.float64)
        scale = np.empty_like(out) if with_scale else None
        rc = lib.oracle_pdf_xfxq2(self._h, len(pids), pids.ctypes.data_as(_ip), n,
                                  x.ctypes.data_as(_dp), q2.ctypes.data_as(_dp),
                                  out.ctypes.data_as(_dp),
                                  scale.ctypes.data_as(_dp) if with_scale else None)
        if rc != 0:
            raise ValueError(f"oracle_pdf_xfxq2 failed with {rc} (requested PID absent?)")
        return (out, scale) if with_scale else out

    @property
    def n_invalid(self) -> int:
        return int(_load().oracle_pdf_grid_invalid(self._h))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.oracle_pdf_grid_free(self._h)
            self._h = None


class OracleAlphas:
    def __init__(self, q_knots, alphas):
        lib = _load()
        q_knots, alphas = _f64(q_knots), _f64(alphas)
        assert q_knots.shape == alphas.shape
        self._h = lib.oracle_alphas_create(len(q_knots), q_knots.ctypes.data_as(_dp),
                                           alphas.ctypes.data_as(_dp))

    @classmethod
    def from_spec(cls, spec):
        return cls(spec.q_knots, spec.alphas)

    def q2(self, q2):
        lib = _load()
        q2 = _f64(np.atleast_1d(q2))
        out = np.empty_like(q2)
        lib.oracle_alphas_q2(self._h, q2.shape[0], q2.ctypes.data_as(_dp), out.ctypes.data_as(_dp))
        return out

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.oracle_alphas_free(self._h)
            self._h = None


def xfxq2_members(x_knots, q_offsets, q_knots, grid_pids, member_values, pids, x, q2, with_scale: bool = False):
    """A PDF set (section 4.3): member m is the single-member interpolation applied
    to member_values[m] on the shared knots -- the definition written out, one member at a time.
    Returns [n_members, n_req, n] (and the scale array of the same shape)."""
    outs, scales = [], []
    for vals in member_values:
        og = OraclePdfGrid(x_knots, q_offsets, q_knots, grid_pids, vals)
        r = og.xfxq2(pids, x, q2, with_scale=with_scale)
        if with_scale:
            outs.append(r[0]); scales.append(r[1])
        else:
            outs.append(r)
    if with_scale:
        return np.stack(outs), np.stack(scales)
    return np.stack(outs)


def lumi_events(og1, terms, x1, x2, q2, og2=None, divide_by_x: bool = False, with_scale: bool = False):
    """Parton luminosity of Monte-Carlo events (x1, x2 and one shared Q^2
    per event): L[e] = sum_t c_t * xf_{a_t}(x1[e], Q2[e]) * xf_{b_t}(x2[e], Q2[e]) -- the definition
    written out: the single-point oracle twice, then the sum over the terms in list order.
    ``og2`` (default: og1) takes the second beam's values from another grid (used by the bilinearity pin).
    with_scale also returns S = sum_t |c_t| (S_a |xf_b| + |xf_a| S_b), the first-order conditioning scale
    of the sum (S_a, S_b the scales of the two factors; tolerance helper only)."""
    og2 = og1 if og2 is None else og2
    terms = [(int(a), int(b), float(c)) for a, b, c in terms]
    pa = sorted({t[0] for t in terms})
    pb = sorted({t[1] for t in terms})
    r1 = og1.xfxq2(pa, x1, q2, with_scale=with_scale)
    r2 = og2.xfxq2(pb, x2, q2, with_scale=with_scale)
    f1, s1 = r1 if with_scale else (r1, None)
    f2, s2 = r2 if with_scale else (r2, None)
    lum = np.zeros(len(np.atleast_1d(x1)), dtype=np.float64)
    sc = np.zeros_like(lum)
    for a, b, c in terms:
        ia, ib = pa.index(a), pb.index(b)
        lum = lum + c * (f1[ia] * f2[ib])
        if with_scale:
            sc = sc + abs(c) * (s1[ia] * np.abs(f2[ib]) + np.abs(f1[ia]) * s2[ib])
    if divide_by_x:
        d = np.asarray(x1, dtype=np.float64) * np.asarray(x2, dtype=np.float64)
        lum = lum / d
        sc = sc / np.abs(d)
    return (lum, sc) if with_scale else lum
