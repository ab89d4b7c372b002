"""Seeded synthetic inputs: knot grids, alpha_s node lists and query batches.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library; it
holds none of the method's arithmetic (no interpolation, no search, no
extrapolation).  It only draws numbers: the analytic value family that fills
the knot grids, the one-loop running coupling that fills the alpha_s nodes, and
the (x, Q^2) query distributions.  It imports neither ``oracle`` nor the CUDA
binding.

The recipes stand in for the paper's benchmark inputs, which are not available
here (NNPDF3.1 NLO grid files; event batches):
"all PDF flavours for an increasingly large number of points distributed
logarithmically in a two-dimensional grid of (x,Q) points, defined within the
boundaries of the original PDF grid".  Shapes follow
BASELINE.json ``configs[0..4]`` (called configs 1-5 below) with the readings
of SURVEY.md section 8(c) Q12-Q14 and 8(d); DESIGN.md restates them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

GRID_SEED = 200906635
PIDS_3 = (1, 2, 21)
PIDS_11 = (-5, -4, -3, -2, -1, 1, 2, 3, 4, 5, 21)
SQRT_S = 13000.0  # GeV, config 5


# --------------------------------------------------------------------------
# containers (plain arrays in the C-ABI's argument layout)
# --------------------------------------------------------------------------
@dataclass
class PdfGridSpec:
    """Host arrays exactly as ``pdf_grid_load`` takes them.

    values has layout [s][ix][iq][ipid] row-major, subgrids concatenated
    (LHAPDF file order).  q_knots are Q in GeV, per subgrid strictly
    increasing, the last of subgrid s equal to the first of subgrid s+1.
    """

    x_knots: np.ndarray
    q_offsets: np.ndarray  # int32, n_sub + 1
    q_knots: np.ndarray
    pids: np.ndarray  # int32
    values: np.ndarray  # flat float64
    params: dict = field(default_factory=dict)  # per-PID (A, a, b, c, d), for tests only
    # per-sub-grid x-knot arrays (LHAPDF allows them): x_knots is then the concatenation, x_offsets
    # (int32, n_sub + 1) delimits the sub-grids' arrays, values are [s][ix_s][iq_s][ipid]
    x_offsets: np.ndarray = None

    @property
    def n_sub(self) -> int:
        return len(self.q_offsets) - 1

    @property
    def nx(self) -> int:
        return len(self.x_knots)

    @property
    def n_pid(self) -> int:
        return len(self.pids)

    def sub_x(self, s: int) -> np.ndarray:
        """x knots of subgrid s."""
        if self.x_offsets is None:
            return self.x_knots
        return self.x_knots[self.x_offsets[s]: self.x_offsets[s + 1]]

    def sub_values(self, s: int) -> np.ndarray:
        """View of subgrid s as [ix][iq][ipid]."""
        off = 0
        for r in range(s):
            off += len(self.sub_x(r)) * int(self.q_offsets[r + 1] - self.q_offsets[r]) * self.n_pid
        nq, nx = int(self.q_offsets[s + 1] - self.q_offsets[s]), len(self.sub_x(s))
        return self.values[off: off + nx * nq * self.n_pid].reshape(nx, nq, self.n_pid)

    def sub_q(self, s: int) -> np.ndarray:
        return self.q_knots[self.q_offsets[s]: self.q_offsets[s + 1]]

    @property
    def q2_min(self) -> float:
        return float(self.q_knots[0] * self.q_knots[0])

    @property
    def q2_max(self) -> float:
        return float(self.q_knots[-1] * self.q_knots[-1])


@dataclass
class AlphasSpec:
    """Host arrays as ``alphas_grid_load`` takes them; a repeated Q marks a threshold."""

    q_knots: np.ndarray
    alphas: np.ndarray


# --------------------------------------------------------------------------
# grid value family  xf = A x^a (1-x)^b (1 + c sqrt x)(1 + d ln(Q^2/2.7))
# --------------------------------------------------------------------------
def draw_family_params(pids, seed: int = GRID_SEED) -> dict:
    """Per PID, in list order: A~U(.5,2), a~U(-.3,.5), b~U(2,6), c~U(-.5,.5), d~U(-.5,.5)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = {}
    for pid in pids:
        A = rng.uniform(0.5, 2.0)
        a = rng.uniform(-0.3, 0.5)
        b = rng.uniform(2.0, 6.0)
        c = rng.uniform(-0.5, 0.5)
        d = rng.uniform(-0.5, 0.5)
        out[int(pid)] = (A, a, b, c, d)
    return out


def family_value(params, x, q2):
    """The analytic family itself (fills knots; tests use it for a gross sanity check)."""
    A, a, b, c, d = params
    x = np.asarray(x, dtype=np.float64)
    q2 = np.asarray(q2, dtype=np.float64)
    return A * x ** a * (1.0 - x) ** b * (1.0 + c * np.sqrt(x)) * (1.0 + d * np.log(q2 / 2.7))


def _geomspace(lo: float, hi: float, n: int) -> np.ndarray:
    k = np.geomspace(lo, hi, n)
    k[0] = lo
    k[-1] = hi
    return k


def make_pdf_grid(x_lo, x_hi, nx, q_edges, nq_per_sub, pids, seed: int = GRID_SEED,
                  sub_scale=None) -> PdfGridSpec:
    """Log-spaced knots, subgrids sharing their edge knot, values from the family.

    ``sub_scale[s]`` multiplies subgrid s (test-only: a jump across thresholds).
    """
    assert len(q_edges) == len(nq_per_sub) + 1
    xk = _geomspace(x_lo, x_hi, nx)
    params = draw_family_params(pids, seed)
    qk, offs, vals = [], [0], []
    for s, nq in enumerate(nq_per_sub):
        q = _geomspace(float(q_edges[s]), float(q_edges[s + 1]), nq)
        qk.append(q)
        offs.append(offs[-1] + nq)
        q2 = q * q
        block = np.empty((nx, nq, len(pids)), dtype=np.float64)
        for k, pid in enumerate(pids):
            block[:, :, k] = family_value(params[int(pid)], xk[:, None], q2[None, :])
        if sub_scale is not None:
            block *= float(sub_scale[s])
        vals.append(block.reshape(-1))
    return PdfGridSpec(
        x_knots=xk,
        q_offsets=np.asarray(offs, dtype=np.int32),
        q_knots=np.concatenate(qk),
        pids=np.asarray(pids, dtype=np.int32),
        values=np.concatenate(vals),
        params=params,
    )


NNPDF_Q_EDGES = (1.65, float(np.sqrt(1.65 * 4.92)), 4.92, 172.5, 1.0e5)
NNPDF_NQ = (7, 14, 23, 20)


def make_pdf_grid_xs(x_knots_per_sub, q_edges, nq_per_sub, pids, seed: int = GRID_SEED) -> PdfGridSpec:
    """A grid whose sub-grids carry their own x-knot arrays (same first and last knot), values from the
    analytic family on each sub-grid's own knots."""
    params = draw_family_params(pids, seed)
    xs = [np.asarray(x, dtype=np.float64) for x in x_knots_per_sub]
    q_offsets, q_knots, vals = [0], [], []
    for s, nq in enumerate(nq_per_sub):
        q = _geomspace(q_edges[s], q_edges[s + 1], nq)
        q_knots.append(q)
        q_offsets.append(q_offsets[-1] + nq)
        blk = np.stack([family_value(params[int(p)], xs[s][:, None], (q * q)[None, :]) for p in pids], axis=-1)
        vals.append(blk.reshape(-1))
    x_off = np.concatenate([[0], np.cumsum([len(x) for x in xs])]).astype(np.int32)
    return PdfGridSpec(np.concatenate(xs), np.asarray(q_offsets, np.int32), np.concatenate(q_knots),
                       np.asarray(pids, np.int32), np.concatenate(vals), params, x_offsets=x_off)


def grid_config1() -> PdfGridSpec:
    """Config 1: 30 x-knots on [1e-6,1], 15 Q-knots on [1.65,100] GeV, PIDs (1,2,21)."""
    return make_pdf_grid(1e-6, 1.0, 30, (1.65, 100.0), (15,), PIDS_3)


def grid_nnpdf_shaped(sub_scale=None) -> PdfGridSpec:
    """Configs 2-5: 100 x-knots on [1e-9,1]; 4 Q subgrids, 7/14/23/20 knots; 11 PIDs."""
    return make_pdf_grid(1e-9, 1.0, 100, NNPDF_Q_EDGES, NNPDF_NQ, PIDS_11, sub_scale=sub_scale)


# --------------------------------------------------------------------------
# PDF sets (Table 2): N_rep member tables on the knots of
# the NNPDF-shaped grid, 13 flavours, evaluated on one x-grid of 2415 points at the fitting scale.
# Stand-in for "N_rep members of NNPDF3.1 NLO" (not available here): member m draws its own
# family parameters from seed GRID_SEED + 7919 * m.
# --------------------------------------------------------------------------
PIDS_13 = (-6, -5, -4, -3, -2, -1, 1, 2, 3, 4, 5, 6, 21)
FK_POINTS = 2415


def grid_member(m: int, pids=PIDS_13) -> PdfGridSpec:
    return make_pdf_grid(1e-9, 1.0, 100, NNPDF_Q_EDGES, NNPDF_NQ, pids, seed=GRID_SEED + 7919 * int(m))


def member_values(n_members: int, pids=PIDS_13, member0: int = 0) -> np.ndarray:
    """[n_members, table size]: each member's values in LHAPDF grid-file order."""
    return np.stack([grid_member(member0 + m, pids).values for m in range(n_members)])


def queries_fk_xgrid(grid: PdfGridSpec, n: int = FK_POINTS, seed: int = 1006):
    """x log-uniform over the grid's x range, all at the lowest scale of the grid (Q0 = 1.65 GeV)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    x = np.clip(_log_uniform(rng, float(grid.x_knots[0]), float(grid.x_knots[-1]), n),
                float(grid.x_knots[0]), float(grid.x_knots[-1]))
    return x, np.full(n, grid.q2_min, dtype=np.float64)


# --------------------------------------------------------------------------
# alpha_s nodes from one-loop running (closed form; used to FILL the grid and
# as a pin for the oracle's interpolation, never as the method)
# --------------------------------------------------------------------------
ALPHAS_MZ = 0.118
MZ = 91.1876
ALPHAS_THRESHOLDS = (1.51, 4.92, 172.5)  # GeV: nf 3|4, 4|5, 5|6
ALPHAS_Q_RANGE = (1.0, 1.0e5)
ALPHAS_NQ = (6, 12, 30, 52)


def _beta0(nf: int) -> float:
    return (33.0 - 2.0 * nf) / (12.0 * np.pi)


def one_loop_alphas(q2):
    """alpha_s(Q^2) at one loop, nf = 3/4/5/6 matched continuously at the thresholds."""
    q2 = np.atleast_1d(np.asarray(q2, dtype=np.float64))
    mc2, mb2, mt2 = (t * t for t in ALPHAS_THRESHOLDS)

    def run(a_ref, mu2_ref, nf, q2_):
        return a_ref / (1.0 + a_ref * _beta0(nf) * np.log(q2_ / mu2_ref))

    a_mb = run(ALPHAS_MZ, MZ * MZ, 5, mb2)
    a_mc = run(a_mb, mb2, 4, mc2)
    a_mt = run(ALPHAS_MZ, MZ * MZ, 5, mt2)
    out = np.empty_like(q2)
    r3 = q2 < mc2
    r4 = (q2 >= mc2) & (q2 < mb2)
    r5 = (q2 >= mb2) & (q2 < mt2)
    r6 = q2 >= mt2
    out[r3] = run(a_mc, mc2, 3, q2[r3])
    out[r4] = run(a_mb, mb2, 4, q2[r4])
    out[r5] = run(ALPHAS_MZ, MZ * MZ, 5, q2[r5])
    out[r6] = run(a_mt, mt2, 6, q2[r6])
    return out


def make_alphas_grid(nq_per_sub=ALPHAS_NQ, q_range=ALPHAS_Q_RANGE,
                     thresholds=ALPHAS_THRESHOLDS, jump=None) -> AlphasSpec:
    """4-subgrid log-spaced node list; ``jump[s]`` scales subgrid s (test-only discontinuity)."""
    edges = (q_range[0],) + tuple(thresholds) + (q_range[1],)
    qs, al = [], []
    for s, nq in enumerate(nq_per_sub):
        q = _geomspace(edges[s], edges[s + 1], nq)
        a = one_loop_alphas(q * q)
        if jump is not None:
            a = a * float(jump[s])
        qs.append(q)
        al.append(a)
    return AlphasSpec(np.concatenate(qs), np.concatenate(al))


# --------------------------------------------------------------------------
# query batches
# --------------------------------------------------------------------------
def _log_uniform(rng, lo: float, hi: float, n: int) -> np.ndarray:
    """exp(U(ln lo, ln hi)) clipped to [lo, hi] (exp can overshoot by an ulp)."""
    v = np.exp(rng.uniform(np.log(lo), np.log(hi), n))
    np.clip(v, lo, hi, out=v)
    return v


def _rng(config: int):
    return np.random.Generator(np.random.PCG64(1000 + config))


def queries_in_range(grid: PdfGridSpec, n: int, config: int, chunk: int = 10_000_000):
    """Configs 1-3: x and Q^2 log-uniform over the grid's own range."""
    rng = _rng(config)
    x = np.empty(n, dtype=np.float64)
    q2 = np.empty(n, dtype=np.float64)
    x_lo, x_hi = float(grid.x_knots[0]), float(grid.x_knots[-1])
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        x[a:b] = _log_uniform(rng, x_lo, x_hi, b - a)
        q2[a:b] = _log_uniform(rng, grid.q2_min, grid.q2_max, b - a)
    return x, q2


def queries_extrapolation_mix(grid: PdfGridSpec, n: int, config: int = 4):
    """Config 4 (reading Q14): 70% in range; 20% x in [1e-12, x_min) with Q^2 in range;
    5% Q in [0.5, Q_min) GeV and 5% Q in (Q_max, 1e6] GeV with x log-uniform on [1e-12, 1];
    randomly permuted."""
    rng = _rng(config)
    x_lo, x_hi = float(grid.x_knots[0]), float(grid.x_knots[-1])
    n_lowx = int(round(0.20 * n))
    n_lowq = int(round(0.05 * n))
    n_highq = int(round(0.05 * n))
    n_in = n - n_lowx - n_lowq - n_highq
    x = np.concatenate([
        _log_uniform(rng, x_lo, x_hi, n_in),
        np.minimum(_log_uniform(rng, 1e-12, x_lo, n_lowx), np.nextafter(x_lo, 0.0)),
        _log_uniform(rng, 1e-12, x_hi, n_lowq),
        _log_uniform(rng, 1e-12, x_hi, n_highq),
    ])
    q_lo, q_hi = float(grid.q_knots[0]), float(grid.q_knots[-1])
    qlow = np.minimum(_log_uniform(rng, 0.5, q_lo, n_lowq), np.nextafter(q_lo, 0.0))
    qhigh = np.maximum(_log_uniform(rng, q_hi, 1.0e6, n_highq), np.nextafter(q_hi, np.inf))
    q2 = np.concatenate([
        _log_uniform(rng, grid.q2_min, grid.q2_max, n_in),
        _log_uniform(rng, grid.q2_min, grid.q2_max, n_lowx),
        qlow * qlow,
        qhigh * qhigh,
    ])
    perm = rng.permutation(n)
    return np.ascontiguousarray(x[perm]), np.ascontiguousarray(q2[perm])


def queries_mc_events(grid: PdfGridSpec, n_events: int, config: int = 5):
    """Config 5: x1, x2 log-uniform on [1e-6,1]; Q^2 = clip(x1 x2 s, q2_min, q2_max)."""
    rng = _rng(config)
    x1 = _log_uniform(rng, 1e-6, 1.0, n_events)
    x2 = _log_uniform(rng, 1e-6, 1.0, n_events)
    q2 = np.clip(x1 * x2 * (SQRT_S * SQRT_S), grid.q2_min, grid.q2_max)
    return x1, x2, q2


def scan_points(grid: PdfGridSpec, per_cell: int = 3):
    """Deterministic scans in the layout of the paper's Fig. 2: every
    x-knot, every Q^2-knot (thresholds included), and ``per_cell`` interior points per
    knot interval, as a full tensor product."""
    xs = [grid.x_knots]
    for f in np.linspace(0.0, 1.0, per_cell + 2)[1:-1]:
        xs.append(grid.x_knots[:-1] ** (1 - f) * grid.x_knots[1:] ** f)
    xs = np.unique(np.clip(np.concatenate(xs), grid.x_knots[0], grid.x_knots[-1]))
    q2k = grid.q_knots * grid.q_knots
    qs = [q2k, np.nextafter(q2k, 0.0)[1:], np.nextafter(q2k, np.inf)[:-1]]
    for s in range(grid.n_sub):
        q = grid.sub_q(s)
        q2s = q * q
        for f in np.linspace(0.0, 1.0, per_cell + 2)[1:-1]:
            qs.append(q2s[:-1] ** (1 - f) * q2s[1:] ** f)
    qs = np.unique(np.clip(np.concatenate(qs), grid.q2_min, grid.q2_max))
    X, Q = np.meshgrid(xs, qs, indexing="ij")
    return np.ascontiguousarray(X.reshape(-1)), np.ascontiguousarray(Q.reshape(-1))


# --------------------------------------------------------------------------
# Writers for the LHAPDF6 text layout (the files themselves are not available here: tests and
# users write synthetic sets with these and read them back through the library's front-end)
# --------------------------------------------------------------------------
def write_lhagrid(spec: PdfGridSpec, path: str, pdf_type: str = "central", x_knots_per_sub=None) -> None:
    """Member file in the LHAPDF6 text layout.  ``x_knots_per_sub`` (a list of x-knot arrays, one per
    sub-grid) writes a file whose sub-grids carry DIFFERENT x knots -- legal in LHAPDF; the library
    reads such a file with pdfb_lhagrid_dims_xs / _get_xs and loads it with pdf_grid_load_xs (the
    one-array entry points pdfb_lhagrid_dims / _get answer PDFB_EXKNOTS); the values of such a block
    are the analytic family of ``spec.params`` on those knots."""
    r = lambda a: " ".join(repr(float(v)) for v in a)
    with open(path, "w") as f:
        f.write(f"PdfType: {pdf_type}\nFormat: lhagrid1\n---\n")
        for s in range(spec.n_sub):
            q = spec.sub_q(s)
            if x_knots_per_sub is None:
                xk = spec.sub_x(s)
                vals = spec.sub_values(s).reshape(len(xk) * len(q), spec.n_pid)
            else:
                xk = np.asarray(x_knots_per_sub[s], dtype=np.float64)
                vals = np.stack([family_value(spec.params[int(p)], xk[:, None], (q * q)[None, :]) for p in spec.pids], axis=-1)
                vals = vals.reshape(len(xk) * len(q), spec.n_pid)
            f.write(r(xk) + "\n" + r(q) + "\n" + " ".join(str(int(p)) for p in spec.pids) + "\n")
            for row in vals:
                f.write(r(row) + "\n")
            f.write("---\n")


def write_lhapdf_info(path: str, n_members: int, pids, alphas_spec) -> None:
    qs = ", ".join(repr(float(v)) for v in alphas_spec.q_knots)
    half = len(alphas_spec.alphas) // 2  # a list that continues on a second line, as real files do
    va = ", ".join(repr(float(v)) for v in alphas_spec.alphas[:half]) + ",\n  " + \
        ", ".join(repr(float(v)) for v in alphas_spec.alphas[half:])
    with open(path, "w") as f:
        f.write(f'SetDesc: "synthetic set written by paper_2009_06635_b200.workloads"\nNumMembers: {int(n_members)}\n')
        f.write("Flavors: [" + ", ".join(str(int(p)) for p in pids) + "]\nFormat: lhagrid1\n")
        f.write(f"AlphaS_Type: ipol\nAlphaS_Qs: [{qs}]\nAlphaS_Vals: [{va}]\n")
