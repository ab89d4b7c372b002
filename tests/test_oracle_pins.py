"""Pins for the CPU oracle (run with -m "not gpu").

The paper prints no worked numeric example for the interpolation (PAPER.md:67-73 give the
method by name only), so the oracle is pinned to what the mathematics fixes: exact knot
reproduction, exactness classes of the scheme, a brute-force evaluation written in a
different form (dense weight matrices), a library routine it must reduce to, the side
rule at thresholds, limits and closed forms of the continuation rules, and the one-loop
alpha_s closed form that fills the alpha_s nodes.  Ids I1-I10 follow SURVEY.md 8(c).
"""
import mpmath
import numpy as np
import pytest
from scipy.interpolate import CubicHermiteSpline

import oracle
from paper_2009_06635_b200 import workloads as W


# ----------------------------------------------------------------------------------
# helpers: tiny hand-made grids and a brute-force evaluator in matrix form
# ----------------------------------------------------------------------------------
def make_spec(xk, q_subs, pids, fn=None, values=None):
    """Grid from explicit knots; fn(s, x[:,None], q2[None,:], pid) -> values."""
    xk = np.asarray(xk, dtype=np.float64)
    offs, vals = [0], []
    for s, q in enumerate(q_subs):
        q = np.asarray(q, dtype=np.float64)
        offs.append(offs[-1] + len(q))
        if values is None:
            blk = np.empty((len(xk), len(q), len(pids)))
            for k, pid in enumerate(pids):
                blk[:, :, k] = fn(s, xk[:, None], (q * q)[None, :], pid)
        else:
            blk = values[s]
        vals.append(np.asarray(blk, dtype=np.float64).reshape(-1))
    return W.PdfGridSpec(xk, np.asarray(offs, np.int32), np.concatenate([np.asarray(q, float) for q in q_subs]),
                         np.asarray(pids, np.int32), np.concatenate(vals))


def fd_matrix(z):
    """M x M matrix of reading O2: one-sided at the ends, mean of one-sided slopes inside."""
    M = len(z)
    D = np.zeros((M, M))
    for m in range(M):
        if m > 0:
            wl = 1.0 if m == M - 1 else 0.5
            D[m, m] += wl / (z[m] - z[m - 1])
            D[m, m - 1] -= wl / (z[m] - z[m - 1])
        if m < M - 1:
            wr = 1.0 if m == 0 else 0.5
            D[m, m + 1] += wr / (z[m + 1] - z[m])
            D[m, m] -= wr / (z[m + 1] - z[m])
    return D


def hbasis(t):
    return (2 * t**3 - 3 * t**2 + 1, t**3 - 2 * t**2 + t, -2 * t**3 + 3 * t**2, t**3 - t**2)


def weights_1d(z, m, zq):
    """Dense weight vector over all knots: value(zq) = w . y for any knot values y."""
    dz = z[m + 1] - z[m]
    t = (zq - z[m]) / dz
    h00, h10, h01, h11 = hbasis(t)
    D = fd_matrix(z)
    w = np.zeros(len(z))
    w[m] += h00
    w[m + 1] += h01
    w += h10 * dz * D[m] + h11 * dz * D[m + 1]
    return w


def locate_py(spec, x, q2):
    s = 0
    for r in range(1, spec.n_sub):
        if spec.sub_q(r)[0] ** 2 <= q2:
            s = r
    xk, q2k = spec.x_knots, spec.sub_q(s) ** 2
    i = int(min(max(np.searchsorted(xk, x, side="right") - 1, 0), len(xk) - 2))
    j = int(min(max(np.searchsorted(q2k, q2, side="right") - 1, 0), len(q2k) - 2))
    return s, i, j


def brute_weights(spec, k, x, q2):
    """sum_ab wu_a wv_b f_ab with dense weight vectors (first form)."""
    s, i, j = locate_py(spec, x, q2)
    U, V = np.log(spec.x_knots), np.log(spec.sub_q(s) ** 2)
    wu, wv = weights_1d(U, i, np.log(x)), weights_1d(V, j, np.log(q2))
    return wu @ spec.sub_values(s)[:, :, k] @ wv


def brute_hermite2d(spec, k, x, q2):
    """Full bicubic Hermite patch on {f, D_u f, D_v f, D_v D_u f} (second form)."""
    s, i, j = locate_py(spec, x, q2)
    U, V = np.log(spec.x_knots), np.log(spec.sub_q(s) ** 2)
    F = spec.sub_values(s)[:, :, k]
    Du, Dv = fd_matrix(U), fd_matrix(V)
    Fu, Fv, Fuv = Du @ F, F @ Dv.T, Du @ F @ Dv.T
    dU, dV = U[i + 1] - U[i], V[j + 1] - V[j]
    hu, hv = hbasis((np.log(x) - U[i]) / dU), hbasis((np.log(q2) - V[j]) / dV)
    val = 0.0
    for a, (ha, hda) in enumerate(((hu[0], hu[1]), (hu[2], hu[3]))):
        for b, (hb, hdb) in enumerate(((hv[0], hv[1]), (hv[2], hv[3]))):
            p, q = i + a, j + b
            val += ha * hb * F[p, q] + dU * hda * hb * Fu[p, q] + dV * ha * hdb * Fv[p, q] \
                + dU * dV * hda * hdb * Fuv[p, q]
    return val


def rand_knots(rng, lo, hi, n):
    k = np.sort(np.exp(rng.uniform(np.log(lo), np.log(hi), n - 2)))
    return np.concatenate([[lo], k, [hi]])


# ----------------------------------------------------------------------------------
# R-ln: the coordinate logarithm is correctly rounded
# ----------------------------------------------------------------------------------
def test_ln_correctly_rounded():
    rng = np.random.default_rng(7)
    xs = np.concatenate([np.exp(rng.uniform(-28, 28, 400)), 1.0 + rng.uniform(-1e-3, 1e-3, 100),
                         [1.0, 2.0, 0.5, 1e-12, 1e10, 2.7]])
    mpmath.mp.prec = 200
    for a in xs:
        assert oracle.ln(float(a)) == float(mpmath.log(mpmath.mpf(float(a))))


# ----------------------------------------------------------------------------------
# I1 knot reproduction
# ----------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["grid1", "grid2"])
def test_I1_knot_reproduction_exact(which, request):
    spec = request.getfixturevalue(which)
    og = oracle.OraclePdfGrid.from_spec(spec)
    for s in range(spec.n_sub):
        q2 = spec.sub_q(s) ** 2
        if s + 1 < spec.n_sub:
            q2 = q2[:-1]  # the threshold knot belongs to the upper subgrid (reading Q2)
        X, Q = np.meshgrid(spec.x_knots, q2, indexing="ij")
        out = og.xfxq2(spec.pids, X.ravel(), Q.ravel())
        ref = spec.sub_values(s)[:, : len(q2), :].transpose(2, 0, 1).reshape(spec.n_pid, -1)
        assert np.array_equal(out, ref)
    assert og.n_invalid == 0


# ----------------------------------------------------------------------------------
# I2 bilinear exactness on non-uniform knots, edge cells and thresholds included
# ----------------------------------------------------------------------------------
def test_I2_bilinear_exact_everywhere_in_range():
    rng = np.random.default_rng(11)
    xk = rand_knots(rng, 1e-5, 1.0, 12)
    qa, qb = rand_knots(rng, 1.3, 4.0, 5), rand_knots(rng, 4.0, 300.0, 7)
    a, b, c, d = 0.7, -0.31, 0.23, 0.045

    def fn(s, x, q2, pid):
        u, v = np.log(x), np.log(q2)
        return a + b * u + c * v + d * u * v

    spec = make_spec(xk, [qa, qb], [21], fn)
    og = oracle.OraclePdfGrid.from_spec(spec)
    x, q2 = W.scan_points(spec, per_cell=4)
    out = og.xfxq2([21], x, q2)[0]
    ref = fn(0, x, q2, 21)
    assert np.max(np.abs(out - ref)) < 2e-14 * np.max(np.abs(ref))


# ----------------------------------------------------------------------------------
# I3 brute force in two other forms on tiny random grids
# ----------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_I3_brute_force_forms_agree(seed):
    rng = np.random.default_rng(seed)
    xk = rand_knots(rng, 1e-4, 1.0, 7)
    subs = [rand_knots(rng, 1.5, 3.0, 2), rand_knots(rng, 3.0, 9.0, 3), rand_knots(rng, 9.0, 200.0, 6)]
    pids = [1, 21]
    values = [rng.normal(size=(len(xk), len(q), len(pids))) for q in subs]
    spec = make_spec(xk, subs, pids, values=values)
    og = oracle.OraclePdfGrid.from_spec(spec)
    x, q2 = W.scan_points(spec, per_cell=2)
    out = og.xfxq2(pids, x, q2)
    scale = max(np.abs(v).max() for v in values)
    for k in range(len(pids)):
        b1 = np.array([brute_weights(spec, k, xi, qi) for xi, qi in zip(x, q2)])
        b2 = np.array([brute_hermite2d(spec, k, xi, qi) for xi, qi in zip(x, q2)])
        assert np.max(np.abs(out[k] - b1)) < 1e-12 * scale
        assert np.max(np.abs(out[k] - b2)) < 1e-12 * scale


# ----------------------------------------------------------------------------------
# I4 quadratics: exact in interior cells, closed-form error in edge cells (pins where
# O2 turns one-sided, i.e. at x edges AND at subgrid thresholds)
# ----------------------------------------------------------------------------------
def test_I4_quadratic_exact_inside_closed_form_error_at_edges():
    nx, nq = 9, 6
    xk = np.exp(np.linspace(np.log(1e-4), 0.0, nx))
    q1 = np.exp(0.5 * np.linspace(np.log(2.0), np.log(30.0), nq))
    q2k = np.exp(0.5 * np.linspace(np.log(30.0), np.log(3000.0), nq))
    q2k[0] = q1[-1]

    def fn(s, x, q2, pid):
        return np.log(x) ** 2 + np.log(q2) ** 2

    spec = make_spec(xk, [q1, q2k], [21], fn)
    og = oracle.OraclePdfGrid.from_spec(spec)
    U = np.log(xk)
    dU = U[1] - U[0]
    x, q2 = W.scan_points(spec, per_cell=3)
    out = og.xfxq2([21], x, q2)[0]
    exact = fn(0, x, q2, 21)
    n_int = n_edge = 0
    for xi, qi, o, e in zip(x, q2, out, exact):
        s, i, j = locate_py(spec, xi, qi)
        V = np.log(spec.sub_q(s) ** 2)
        dV = V[1] - V[0]
        t, tau = (np.log(xi) - U[i]) / dU, (np.log(qi) - V[j]) / dV
        # one-sided slope of a parabola is off by +-Delta; that derivative enters through
        # h10 (left knot) or h11 (right knot), times the interval length
        err = 0.0
        if i == 0:
            err += dU * dU * hbasis(t)[1]
        if i == nx - 2:
            err -= dU * dU * hbasis(t)[3]
        if j == 0:
            err += dV * dV * hbasis(tau)[1]
        if j == nq - 2:
            err -= dV * dV * hbasis(tau)[3]
        assert abs((o - e) - err) < 1e-11 * max(1.0, abs(e)), (s, i, j)
        if err == 0.0:
            n_int += 1
        elif abs(err) > 1e-3:
            n_edge += 1
    assert n_int > 100 and n_edge > 100


# ----------------------------------------------------------------------------------
# I5 library special case: constant in Q -> scipy CubicHermiteSpline in u (and vice versa)
# ----------------------------------------------------------------------------------
def test_I5_reduces_to_scipy_cubic_hermite_spline():
    rng = np.random.default_rng(5)
    xk = rand_knots(rng, 1e-6, 1.0, 15)
    qk = rand_knots(rng, 1.5, 500.0, 9)
    gx, gq = rng.normal(size=len(xk)), rng.normal(size=len(qk))
    U, V = np.log(xk), np.log(qk * qk)
    spec = make_spec(xk, [qk], [1, 2], values=[np.stack(
        [np.repeat(gx[:, None], len(qk), 1), np.repeat(gq[None, :], len(xk), 0)], axis=-1)])
    og = oracle.OraclePdfGrid.from_spec(spec)
    x, q2 = W.scan_points(spec, per_cell=3)
    out = og.xfxq2([1, 2], x, q2)
    sx = CubicHermiteSpline(U, gx, fd_matrix(U) @ gx)
    sq = CubicHermiteSpline(V, gq, fd_matrix(V) @ gq)
    assert np.max(np.abs(out[0] - sx(np.log(x)))) < 5e-14
    assert np.max(np.abs(out[1] - sq(np.log(q2)))) < 5e-14


# ----------------------------------------------------------------------------------
# I6 threshold side rule
# ----------------------------------------------------------------------------------
def test_I6_threshold_point_uses_upper_subgrid():
    spec = W.grid_nnpdf_shaped(sub_scale=(1.0, 1.01, 1.0201, 1.030301))
    og = oracle.OraclePdfGrid.from_spec(spec)
    x = spec.x_knots[10:60:7]
    for s in range(1, spec.n_sub):
        qth = spec.sub_q(s)[0] ** 2
        assert qth == spec.sub_q(s - 1)[-1] ** 2
        up = og.xfxq2(spec.pids, x, np.full_like(x, qth))
        lo = og.xfxq2(spec.pids, x, np.full_like(x, np.nextafter(qth, 0.0)))
        ref_up = spec.sub_values(s)[10:60:7, 0, :].T
        ref_lo = spec.sub_values(s - 1)[10:60:7, -1, :].T
        assert np.array_equal(up, ref_up)
        assert np.allclose(lo, ref_lo, rtol=1e-13, atol=1e-13)
        assert np.all(np.abs(up - lo) > 5e-3 * np.abs(ref_lo))  # the 1% jump is seen


def test_derivatives_do_not_cross_thresholds():
    """Rows j-1 / j+2 are never taken from a neighbouring subgrid: changing subgrid s+1
    cannot change any value in subgrid s."""
    a = W.grid_nnpdf_shaped()
    b = W.grid_nnpdf_shaped(sub_scale=(1.0, 1.0, 3.0, 1.0))
    oa, ob = oracle.OraclePdfGrid.from_spec(a), oracle.OraclePdfGrid.from_spec(b)
    x, q2 = W.queries_in_range(a, 4000, 2)
    lo, hi = a.sub_q(2)[0] ** 2, a.sub_q(2)[-1] ** 2
    outside = (q2 < lo) | (q2 >= hi)
    va, vb = oa.xfxq2(a.pids, x, q2), ob.xfxq2(b.pids, x, q2)
    assert np.array_equal(va[:, outside], vb[:, outside])
    assert np.allclose(3.0 * va[:, ~outside], vb[:, ~outside], rtol=1e-12, atol=1e-13)


# ----------------------------------------------------------------------------------
# I7 continuity of the continuation rules at the grid border
# ----------------------------------------------------------------------------------
def test_I7_continuation_is_continuous_at_the_border(grid2, ograph2):
    pids = grid2.pids
    x0, xm = grid2.x_knots[0], 3.3e-4
    qmin, qmax = grid2.q2_min, grid2.q2_max
    qmid = 77.0
    eps = 1e-9
    # A: x -> x0 from below
    a_in = ograph2.xfxq2(pids, [x0], [qmid])
    a_out = ograph2.xfxq2(pids, [x0 * (1 - eps)], [qmid])
    assert np.allclose(a_in, a_out, rtol=1e-7, atol=1e-9)
    # B: Q^2 -> qmax from above;  C: Q^2 -> qmin from below
    for x in (xm, x0 * 0.5):
        b_in = ograph2.xfxq2(pids, [x], [qmax])
        b_out = ograph2.xfxq2(pids, [x], [qmax * (1 + eps)])
        assert np.allclose(b_in, b_out, rtol=1e-7, atol=1e-9)
        c_in = ograph2.xfxq2(pids, [x], [qmin])
        c_out = ograph2.xfxq2(pids, [x], [qmin * (1 - eps)])
        assert np.allclose(c_in, c_out, rtol=1e-6, atol=1e-9)


# ----------------------------------------------------------------------------------
# I8 closed forms of the continuation
# ----------------------------------------------------------------------------------
def _powerlaw_spec(A=2.0, a=-0.25, g=0.15, nq=10):
    xk = np.geomspace(1e-5, 1.0, 14)
    qk = np.geomspace(2.0, 1000.0, nq)

    def fn(s, x, q2, pid):
        return A * x**a * q2**g

    return make_spec(xk, [qk], [21], fn), (A, a, g)


def test_I8_rule_A_and_B_are_exact_power_laws():
    spec, (A, a, g) = _powerlaw_spec()
    og = oracle.OraclePdfGrid.from_spec(spec)
    x0, q2lo, q2hi = spec.x_knots[0], spec.q2_min, spec.q2_max
    # A: below x0 the value continues as (x/x0)^a from the border value
    xs = x0 * np.array([0.9, 0.3, 1e-2, 1e-5])
    qs = np.full_like(xs, 57.0)
    border = og.xfxq2([21], [x0], [57.0])[0, 0]
    got = og.xfxq2([21], xs, qs)[0]
    assert np.allclose(got, border * (xs / x0) ** a, rtol=2e-13)
    # B: above q_max the value continues with the log-slope of the last two knots, = g
    Qs = q2hi * np.array([1.5, 10.0, 1e3])
    for x in (3e-3, x0 * 0.1):
        edge = og.xfxq2([21], [x], [q2hi])[0, 0]
        got = og.xfxq2([21], np.full_like(Qs, x), Qs)[0]
        assert np.allclose(got, edge * (Qs / q2hi) ** g, rtol=2e-13)
    # corner value = A x^a Q2^g itself (both rules are exact for a pure power law at knots)
    got = og.xfxq2([21], [x0 * 0.01], [q2hi * 100.0])[0, 0]
    assert np.isclose(got, A * (x0 * 0.01) ** a * (q2hi * 100.0) ** g, rtol=1e-12)
    assert og.n_invalid == 0


def test_I8_small_values_continue_linearly_in_log():
    """Values <= 1e-3 (or negative): the log-lin branch is a straight line in ln x / ln Q^2."""
    xk = np.geomspace(1e-4, 1.0, 9)
    qk = np.geomspace(2.0, 100.0, 6)
    c0, c1, c2 = 2e-4, 1.5e-5, -2.0e-5

    def fn(s, x, q2, pid):
        return c0 + c1 * np.log(x) + c2 * np.log(q2)

    spec = make_spec(xk, [qk], [21], fn)
    assert spec.values.max() < 1e-3
    og = oracle.OraclePdfGrid.from_spec(spec)
    xs = np.array([5e-5, 1e-6, 1e-9, 3e-3, 1e-7])
    qs = np.array([30.0, 8.0, 2.0e4, 5.0e5, 9.9e6])  # A, A, B, B, corner A+B
    got = og.xfxq2([21], xs, qs)[0]
    assert np.allclose(got, fn(0, xs, qs, 21), rtol=0, atol=1e-17)


def test_I8_rule_C_limits_clamp_and_fallback():
    spec, (A, a, g) = _powerlaw_spec(g=0.4)
    og = oracle.OraclePdfGrid.from_spec(spec)
    qmin = spec.q2_min
    x = spec.x_knots[5]
    y0 = og.xfxq2([21], [x], [qmin])[0, 0]
    y1 = og.xfxq2([21], [x], [1.01 * qmin])[0, 0]
    gamma = (y1 - y0) / y0 / 0.01
    # anomalous dimension ~ log-slope of the interpolant at q_min = secant slope of the
    # first Q^2 interval (one-sided rule at the subgrid edge)
    ratio = (spec.q_knots[1] / spec.q_knots[0]) ** 2
    assert abs(gamma - (ratio ** g - 1.0) / np.log(ratio)) < 0.01
    # (i) just below q_min the log-slope equals gamma
    r1, r2 = 1 - 1e-4, 1 - 2e-4
    f1, f2 = og.xfxq2([21], [x, x], [r1 * qmin, r2 * qmin])[0]
    assert abs((np.log(f1) - np.log(f2)) / (np.log(r1) - np.log(r2)) - gamma) < 2e-3
    # (ii) far below q_min xf vanishes linearly in Q^2: f / rho -> y0
    rho = 1e-7
    f = og.xfxq2([21], [x], [rho * qmin])[0, 0]
    assert abs(f / rho / y0 - 1.0) < 1e-4
    # (iii) closed form at one mid point
    rho = 0.37
    f = og.xfxq2([21], [x], [rho * qmin])[0, 0]
    assert np.isclose(f, y0 * rho ** (gamma * rho + 1 - rho), rtol=1e-13)
    # (iv) clamp: a grid falling steeply towards larger Q^2 has gamma_raw < -2.5
    spec2, _ = _powerlaw_spec(A=2000.0, g=-8.0, nq=40)
    og2 = oracle.OraclePdfGrid.from_spec(spec2)
    y0 = og2.xfxq2([21], [x], [qmin])[0, 0]
    y1 = og2.xfxq2([21], [x], [1.01 * qmin])[0, 0]
    assert abs(y0) > 1e-5 and (y1 - y0) / y0 / 0.01 < -2.6
    f = og2.xfxq2([21], [x], [0.5 * qmin])[0, 0]
    assert np.isclose(f, y0 * 0.5 ** (-2.5 * 0.5 + 0.5), rtol=1e-13)
    # (v) |y0| < 1e-5 -> gamma = 1: the exponent gamma*rho + 1 - rho is 1 for every rho, so xf is
    # the straight line y0 * Q^2/q_min through the origin -- the limit (ii) that the regular branch
    # reaches as rho -> 0, now at every rho (reading Q9)
    spec3, _ = _powerlaw_spec(A=1e-6, g=0.4)
    og3 = oracle.OraclePdfGrid.from_spec(spec3)
    y0 = og3.xfxq2([21], [0.5], [qmin])[0, 0]
    assert 0 < abs(y0) < 1e-5
    rhos = np.array([0.9, 0.5, 0.1, 1e-3])
    f = og3.xfxq2([21], np.full_like(rhos, 0.5), rhos * qmin)[0]
    assert np.allclose(f, y0 * rhos, rtol=2e-15, atol=0)
    assert np.allclose(np.diff(f) / np.diff(rhos), y0, rtol=1e-12)  # one slope: a straight line


def _two_column_spec(yL, yH, qk=None):
    """Grid constant along Q whose first two x columns hold yL, yH (values given explicitly)."""
    xk = np.geomspace(1e-4, 1.0, 7)
    qk = np.geomspace(2.0, 100.0, 6) if qk is None else qk
    col = np.array([yL, yH, 0.5, 0.4, 0.3, 0.2, 0.0])
    vals = np.repeat(col[:, None], len(qk), axis=1)[:, :, None]
    return make_spec(xk, [qk], [21], values=[vals])


@pytest.mark.parametrize("yL,loglog", [(1.001e-3, True), (0.999e-3, False), (1e-3, False)])
def test_I8_O4_switches_at_1e_minus_3(yL, loglog):
    """O4 is linear in log-log iff BOTH values are strictly above 1e-3, else linear in log-lin:
    pinned 0.1 % either side of the switch and exactly on it (closed forms written out here)."""
    yH = 1.3e-3
    spec = _two_column_spec(yL, yH)
    og = oracle.OraclePdfGrid.from_spec(spec)
    x0, x1 = spec.x_knots[0], spec.x_knots[1]
    q2 = float(spec.q_knots[2]) ** 2          # on a Q^2 knot: the two probes are yL, yH exactly
    xs = x0 * np.array([0.5, 1e-2, 1e-6])
    r = np.log(xs / x0) / np.log(x1 / x0)
    got = og.xfxq2([21], xs, np.full_like(xs, q2))[0]
    power = yL * (yH / yL) ** r
    line = yL + r * (yH - yL)
    assert np.all(np.abs(power - line) > 1e-6)  # the two branches are far apart at these points
    assert np.allclose(got, power if loglog else line, rtol=1e-13, atol=0)
    # the same switch with the roles swapped (yH at the threshold)
    spec = _two_column_spec(1.3e-3, yL)
    got = oracle.OraclePdfGrid.from_spec(spec).xfxq2([21], xs, np.full_like(xs, q2))[0]
    power, line = 1.3e-3 * (yL / 1.3e-3) ** r, 1.3e-3 + r * (yL - 1.3e-3)
    assert np.allclose(got, power if loglog else line, rtol=1e-13, atol=0)


@pytest.mark.parametrize("y0,regular", [(1.001e-5, True), (0.999e-5, False), (1e-5, True), (-1.001e-5, True), (-0.999e-5, False)])
def test_I8_O5C_fallback_switches_at_1e_minus_5(y0, regular):
    """Rule C takes gamma from the probe at 1.01 q_min iff |y0| >= 1e-5, else gamma = 1."""
    xk = np.geomspace(1e-4, 1.0, 7)
    qk = np.geomspace(2.0, 100.0, 6)
    g = 0.3
    row = (qk * qk / qk[0] ** 2) ** g
    vals = np.empty((len(xk), len(qk), 1))
    vals[:, :, 0] = y0 * row[None, :]
    vals[:, 0, 0] = y0                      # the q_min row holds y0 exactly
    spec = make_spec(xk, [qk], [21], values=[vals])
    og = oracle.OraclePdfGrid.from_spec(spec)
    x, qmin = float(xk[3]), spec.q2_min
    assert og.xfxq2([21], [x], [qmin])[0, 0] == y0
    y1 = og.xfxq2([21], [x], [1.01 * qmin])[0, 0]
    gamma = max(-2.5, (y1 - y0) / y0 / 0.01)
    assert 0.2 < gamma < 0.4                # far from 1: the two branches differ visibly
    rho = np.array([0.8, 0.3, 0.05])
    got = og.xfxq2([21], np.full_like(rho, x), rho * qmin)[0]
    want = y0 * rho ** (gamma * rho + 1 - rho) if regular else y0 * rho
    assert np.allclose(got, want, rtol=1e-13, atol=0)


def test_invalid_points_give_nan_and_are_counted(grid1):
    og = oracle.OraclePdfGrid.from_spec(grid1)
    x = np.array([0.5, 1.0000001, 0.0, -0.1, np.nan, 0.5, 0.5, 0.5])
    q2 = np.array([10.0, 10.0, 10.0, 10.0, 10.0, 0.0, -3.0, np.nan])
    out = og.xfxq2(grid1.pids, x, q2)
    assert np.all(np.isfinite(out[:, 0])) and np.all(np.isnan(out[:, 1:]))
    assert og.n_invalid == 7


def test_pid_alias_and_unknown_pid(grid1, ograph1):
    x, q2 = W.queries_in_range(grid1, 100, 1)
    assert np.array_equal(ograph1.xfxq2([0], x, q2), ograph1.xfxq2([21], x, q2))
    assert np.array_equal(ograph1.xfxq2([21, 1], x, q2)[1], ograph1.xfxq2([1], x, q2)[0])
    with pytest.raises(ValueError):
        ograph1.xfxq2([6], x, q2)


# ----------------------------------------------------------------------------------
# I10 gross sanity against the analytic family
# ----------------------------------------------------------------------------------
def test_I10_close_to_the_analytic_family(grid2, ograph2):
    x, q2 = W.queries_in_range(grid2, 20000, 2)
    out = ograph2.xfxq2(grid2.pids, x, q2)
    away = x < grid2.x_knots[-3]
    for k, pid in enumerate(grid2.pids):
        ana = W.family_value(grid2.params[int(pid)], x, q2)
        rel = np.abs(out[k] - ana) / (np.abs(ana) + 1e-3)
        assert np.median(rel) < 1e-4
        assert rel[away].max() < 5e-2


# ----------------------------------------------------------------------------------
# I9 alpha_s
# ----------------------------------------------------------------------------------
def test_I9_alphas_matches_one_loop_and_converges():
    """Within 1e-3 of the closed form on the config-5 node list; halving the spacing cuts
    the error 8x in interior cells (O(h^3): mean-of-slopes derivative is O(h^2) accurate)
    and 4x in subgrid-edge cells (one-sided derivative, O(h) accurate)."""
    e_int, e_edge = [], []
    for mult in (1, 2, 4):
        nq = tuple(mult * (n - 1) + 1 for n in W.ALPHAS_NQ)
        spec = W.make_alphas_grid(nq)
        oa = oracle.OracleAlphas.from_spec(spec)
        rng = np.random.default_rng(3)
        q2 = np.exp(rng.uniform(np.log(1.0), np.log(1e10), 50000))
        got, ref = oa.q2(q2), W.one_loop_alphas(q2)
        rel = np.abs(got - ref) / ref
        edge = np.zeros(len(q2), dtype=bool)
        off = np.cumsum((0,) + nq)
        for s in range(4):
            k2 = spec.q_knots[off[s]:off[s + 1]] ** 2
            edge |= ((q2 >= k2[0]) & (q2 < k2[1])) | ((q2 >= k2[-2]) & (q2 <= k2[-1]))
        e_int.append(rel[~edge].max())
        e_edge.append(rel[edge].max())
        if mult == 1:
            kq2 = spec.q_knots ** 2
            keep = np.concatenate([kq2[1:] != kq2[:-1], [True]])  # threshold -> upper node
            assert np.array_equal(oa.q2(kq2[keep]), spec.alphas[keep])
    assert max(e_int[0], e_edge[0]) < 1e-3
    assert e_int[0] / e_int[1] > 6.5 and e_int[1] / e_int[2] > 6.5
    assert 3.5 < e_edge[0] / e_edge[1] < 5.0 and 3.5 < e_edge[1] / e_edge[2] < 5.0


def test_alphas_constant_outside_and_threshold_side():
    spec = W.make_alphas_grid(jump=(1.0, 1.02, 1.0404, 1.061208))
    oa = oracle.OracleAlphas.from_spec(spec)
    q2lo, q2hi = spec.q_knots[0] ** 2, spec.q_knots[-1] ** 2
    assert np.array_equal(oa.q2([q2lo * 0.5, q2lo * 1e-6, q2hi * 2, q2hi * 1e8]),
                          [spec.alphas[0]] * 2 + [spec.alphas[-1]] * 2)
    assert np.isnan(oa.q2([0.0, -1.0, np.nan])).all()
    off = np.cumsum((0,) + W.ALPHAS_NQ)
    for s in range(1, 4):
        qth = spec.q_knots[off[s]] ** 2
        assert oa.q2([qth])[0] == spec.alphas[off[s]]
        below = oa.q2([np.nextafter(qth, 0.0)])[0]
        assert np.isclose(below, spec.alphas[off[s] - 1], rtol=1e-13)
        assert abs(below - spec.alphas[off[s]]) > 0.01 * below


def test_alphas_single_subgrid_is_scipy_hermite():
    rng = np.random.default_rng(9)
    q = rand_knots(rng, 1.0, 1e4, 17)
    a = 0.1 + 0.05 * rng.random(17)
    oa = oracle.OracleAlphas(q, a)
    Z = np.log(q * q)
    sp = CubicHermiteSpline(Z, a, fd_matrix(Z) @ a)
    q2 = np.exp(rng.uniform(Z[0], Z[-1], 5000))
    assert np.max(np.abs(oa.q2(q2) - sp(np.log(q2)))) < 1e-15


# ----------------------------------------------------------------------------------
# conditioning scale (tolerance helper) bounds the weighted stencil magnitude
# ----------------------------------------------------------------------------------
def test_scale_bounds_weighted_stencil_sum():
    rng = np.random.default_rng(4)
    xk = rand_knots(rng, 1e-4, 1.0, 8)
    subs = [rand_knots(rng, 1.5, 9.0, 4), rand_knots(rng, 9.0, 200.0, 5)]
    values = [rng.normal(size=(len(xk), len(q), 1)) for q in subs]
    spec = make_spec(xk, subs, [21], values=values)
    og = oracle.OraclePdfGrid.from_spec(spec)
    x, q2 = W.scan_points(spec, per_cell=2)
    out, scale = og.xfxq2([21], x, q2, with_scale=True)
    for xi, qi, o, sc in zip(x[::7], q2[::7], out[0, ::7], scale[0, ::7]):
        s, i, j = locate_py(spec, xi, qi)
        U, V = np.log(spec.x_knots), np.log(spec.sub_q(s) ** 2)
        wu, wv = weights_1d(U, i, np.log(xi)), weights_1d(V, j, np.log(qi))
        S = np.abs(wu) @ np.abs(spec.sub_values(s)[:, :, 0]) @ np.abs(wv)
        assert sc >= S * (1 - 1e-12) and sc <= 8 * S + 1e-300
        assert abs(o) <= sc * (1 + 1e-12)


@pytest.mark.parametrize("kind", ["loglog", "loglin", "tiny"])
def test_scale_bounds_the_sensitivity_outside_the_grid(kind):
    """The scale helper outside the grid (cont_scale, G_scale, the Q^2 < q_min and Q^2 > q_max
    branches of xf_scale) against what it claims to bound: S = sum_knots |d result / d f_knot| |f_knot|,
    the derivatives taken numerically by perturbing one table value at a time.  Classes A, B, C
    and both corners; grids whose values take O4's log-log branch, its log-lin branch, and rule C's
    |y0| < 1e-5 branch."""
    rng = np.random.default_rng(11 if kind == "loglog" else 12)
    xk = rand_knots(rng, 1e-4, 1.0, 5)
    subs = [rand_knots(rng, 1.5, 9.0, 4), rand_knots(rng, 9.0, 200.0, 4)]
    if kind == "loglog":   # all values >> 1e-3
        values = [np.exp(0.3 * rng.normal(size=(len(xk), len(q), 1))) for q in subs]
    else:                  # all |values| < 1e-3, both signs; "tiny": |y0| < 1e-5, rule C's gamma = 1 branch
        amp = 2e-4 if kind == "loglin" else 2e-6
        values = [amp * rng.normal(size=(len(xk), len(q), 1)) for q in subs]
    spec = make_spec(xk, subs, [21], values=values)
    x0, xm = spec.x_knots[0], 0.37 * spec.x_knots[2] + 0.63 * spec.x_knots[3]
    qlo, qhi, qmid = spec.q2_min, spec.q2_max, 30.0
    pts = np.array([(0.3 * x0, qmid), (1e-3 * x0, 4.0),          # A
                    (xm, 3.0 * qhi), (xm, 1e3 * qhi),            # B
                    (xm, 0.6 * qlo), (xm, 0.05 * qlo),           # C
                    (0.2 * x0, 7.0 * qhi), (0.2 * x0, 0.4 * qlo)])  # corners A+B, A+C
    x, q2 = pts[:, 0].copy(), pts[:, 1].copy()
    base, scale = oracle.OraclePdfGrid.from_spec(spec).xfxq2([21], x, q2, with_scale=True)
    flat = spec.values.copy()
    S = np.zeros(len(x))
    for e in range(len(flat)):
        d = 1e-6 * abs(flat[e])
        hi, lo = flat.copy(), flat.copy()
        hi[e] += d; lo[e] -= d
        fh = oracle.OraclePdfGrid(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, hi).xfxq2([21], x, q2)[0]
        fl = oracle.OraclePdfGrid(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, lo).xfxq2([21], x, q2)[0]
        S += np.abs(fh - fl) / (2 * d) * abs(flat[e])
    assert np.all(S > 0)
    assert np.all(scale[0] >= S * (1 - 1e-6)), (scale[0] / S)
    assert np.all(scale[0] <= 400 * S), (scale[0] / S)   # a bound, not a blank cheque
    assert np.all(np.abs(base[0]) <= scale[0] * (1 + 1e-12))


# ----------------------------------------------------------------------------------
# PDF sets: the member helper is the single-member interpolation per table;
# pinned by what the mathematics fixes -- in range the interpolant is LINEAR in the table values
# ----------------------------------------------------------------------------------
def test_member_set_is_linear_in_the_tables():
    rng = np.random.default_rng(41)
    xk = rand_knots(rng, 1e-5, 1.0, 9)
    subs = [rand_knots(rng, 1.5, 4.0, 5), rand_knots(rng, 4.0, 90.0, 6)]
    pids = [1, 2, 21]
    size = sum(len(xk) * len(q) * len(pids) for q in subs)
    f1, f2 = rng.normal(size=size), rng.normal(size=size)
    a, b = 0.75, -2.5
    spec = make_spec(xk, subs, pids, values=[np.zeros((len(xk), len(q), len(pids))) for q in subs])
    x, q2 = W.scan_points(spec, per_cell=4)
    tabs = np.stack([f1, f2, a * f1 + b * f2])
    out, sc = oracle.xfxq2_members(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, tabs, pids, x, q2,
                                   with_scale=True)
    assert out.shape == (3, len(pids), len(x))
    lin = a * out[0] + b * out[1]
    S = abs(a) * sc[0] + abs(b) * sc[1]
    assert np.all(np.abs(out[2] - lin) <= 8e-16 * S + 1e-300), np.max(np.abs(out[2] - lin) / S)
    # and each member is exactly the single-member oracle on its own table
    for m in range(3):
        single = oracle.OraclePdfGrid(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, tabs[m]).xfxq2(pids, x, q2)
        assert np.array_equal(single, out[m])


# ----------------------------------------------------------------------------------
# Parton luminosity of events: the helper is "the single-point oracle
# twice, then the sum over the terms"; pinned by what the mathematics fixes -- in range it is
# BILINEAR in the tables of the two beams, a single term is the product of two single values, and
# exchanging the beams together with the pair table changes nothing.
# ----------------------------------------------------------------------------------
def test_lumi_helper_is_bilinear_and_symmetric():
    rng = np.random.default_rng(43)
    xk = rand_knots(rng, 1e-5, 1.0, 9)
    subs = [rand_knots(rng, 1.5, 4.0, 5), rand_knots(rng, 4.0, 90.0, 6)]
    pids = [-1, 1, 2, 21]
    size = sum(len(xk) * len(q) * len(pids) for q in subs)
    spec = make_spec(xk, subs, pids, values=[np.zeros((len(xk), len(q), len(pids))) for q in subs])

    def og(tab):
        return oracle.OraclePdfGrid(spec.x_knots, spec.q_offsets, spec.q_knots, spec.pids, tab)

    t1, t2, t3 = rng.normal(size=size), rng.normal(size=size), rng.normal(size=size)
    a, b = 0.5, -1.75
    n = 400
    x1 = np.exp(rng.uniform(np.log(xk[0]), 0.0, n)); x2 = np.exp(rng.uniform(np.log(xk[0]), 0.0, n))
    q2 = np.exp(rng.uniform(np.log(spec.q2_min), np.log(spec.q2_max), n))
    terms = [(1, -1, 1.0), (-1, 1, 1.0), (21, 21, 0.3), (2, 0, -0.7), (2, 21, 0.1)]   # PID 0 = 21; (2,21) appears twice
    L = lambda g1, g2: oracle.lumi_events(g1, terms, x1, x2, q2, og2=g2, with_scale=True)
    l13, s13 = L(og(t1), og(t3)); l23, s23 = L(og(t2), og(t3)); lc3, _ = L(og(a * t1 + b * t2), og(t3))
    assert np.all(np.abs(lc3 - (a * l13 + b * l23)) <= 4e-15 * (abs(a) * s13 + abs(b) * s23) + 1e-300)
    l31, s31 = L(og(t3), og(t1)); l32, s32 = L(og(t3), og(t2)); l3c, _ = L(og(t3), og(a * t1 + b * t2))
    assert np.all(np.abs(l3c - (a * l31 + b * l32)) <= 4e-15 * (abs(a) * s31 + abs(b) * s32) + 1e-300)
    # one term with unit coefficient = the product of the two single-point values, bit for bit
    g1 = og(t1)
    single = oracle.lumi_events(g1, [(2, -1, 1.0)], x1, x2, q2)
    assert np.array_equal(single, g1.xfxq2([2], x1, q2)[0] * g1.xfxq2([-1], x2, q2)[0])
    # exchanging the beams and transposing the pair table changes nothing but the summation order
    swapped = oracle.lumi_events(g1, [(b_, a_, c) for a_, b_, c in terms], x2, x1, q2)
    direct, sc = oracle.lumi_events(g1, terms, x1, x2, q2, with_scale=True)
    assert np.all(np.abs(swapped - direct) <= 4e-16 * sc + 1e-300)
    # the 1/(x1 x2) form, and the scale bounds the sum of term magnitudes
    assert np.allclose(oracle.lumi_events(g1, terms, x1, x2, q2, divide_by_x=True), direct / (x1 * x2), rtol=4e-16, atol=0)
    assert np.all(np.abs(direct) <= sc * (1 + 1e-12))


# ----------------------------------------------------------------------------------
# Per-sub-grid x-knot arrays (the LHAPDF layout allows them; "computes independently query
# points belonging to different sub-grids"): a sub-grid with its own x knots is interpolated exactly
# as if it were a grid of its own.
# ----------------------------------------------------------------------------------
def test_per_subgrid_x_knots_are_independent_grids():
    rng = np.random.default_rng(51)
    subs = [rand_knots(rng, 1.5, 4.0, 5), rand_knots(rng, 4.0, 30.0, 6), rand_knots(rng, 30.0, 900.0, 4)]
    xs = [rand_knots(rng, 1e-5, 1.0, n) for n in (9, 14, 6)]
    pids = [1, 21]
    vals = [rng.normal(size=(len(x), len(q), len(pids))) for x, q in zip(xs, subs)]
    x_off = np.concatenate([[0], np.cumsum([len(x) for x in xs])]).astype(np.int32)
    q_off = np.concatenate([[0], np.cumsum([len(q) for q in subs])]).astype(np.int32)
    og = oracle.OraclePdfGrid(np.concatenate(xs), q_off, np.concatenate(subs), pids,
                              np.concatenate([v.reshape(-1) for v in vals]), x_offsets=x_off)
    for s, (xk, qk, v) in enumerate(zip(xs, subs, vals)):
        single = oracle.OraclePdfGrid(xk, [0, len(qk)], qk, pids, v.reshape(-1))
        lo, hi = qk[0] ** 2, qk[-1] ** 2
        n = 500
        x = np.exp(rng.uniform(np.log(1e-7), 0.0, n))                       # in range and below x_0 (rule A)
        x[:len(xk)] = xk
        q2 = np.exp(rng.uniform(np.log(lo), np.log(hi), n))
        q2 = np.clip(q2, lo, np.nextafter(hi, 0) if s + 1 < len(subs) else hi)  # the threshold itself belongs to s + 1
        a, sa = og.xfxq2(pids, x, q2, with_scale=True)
        b, sb = single.xfxq2(pids, x, q2, with_scale=True)
        assert np.array_equal(a, b) and np.array_equal(sa, sb)
    # knots of every sub-grid are reproduced exactly, thresholds in the upper sub-grid
    for s, (xk, qk, v) in enumerate(zip(xs, subs, vals)):
        qq = qk[:-1] if s + 1 < len(subs) else qk
        X, Q = np.meshgrid(xk, qq ** 2, indexing="ij")
        got = og.xfxq2(pids, X.ravel(), Q.ravel())
        assert np.array_equal(got, v[:, :len(qq), :].transpose(2, 0, 1).reshape(len(pids), -1))
    # one shared array passed sub-grid by sub-grid = the shared-array form, bit for bit
    xk = xs[0]
    vals2 = [rng.normal(size=(len(xk), len(q), len(pids))) for q in subs]
    flat = np.concatenate([v.reshape(-1) for v in vals2])
    shared = oracle.OraclePdfGrid(xk, q_off, np.concatenate(subs), pids, flat)
    per = oracle.OraclePdfGrid(np.tile(xk, 3), q_off, np.concatenate(subs), pids, flat,
                               x_offsets=np.arange(4, dtype=np.int32) * len(xk))
    x = np.exp(rng.uniform(np.log(1e-7), 0.0, 2000)); q2 = np.exp(rng.uniform(np.log(0.5), np.log(2e6), 2000))
    assert np.array_equal(shared.xfxq2(pids, x, q2), per.xfxq2(pids, x, q2), equal_nan=True)


def test_C1_inside_a_subgrid_and_a_kink_only_at_thresholds():
    """A cubic Hermite interpolant with ONE derivative per knot (reading O2) is C1: along either axis the
    slope just left of an interior knot equals the slope just right of it, on random non-uniform knots
    and random values.  Across a Q^2 threshold the sub-grids are interpolated independently (P2), so
    there -- and only there -- the slope may jump.  (A derivative rule that differs between the two
    cells sharing a knot, or a stencil shifted by one, shows up as a kink of order 1.)"""
    rng = np.random.default_rng(42)
    xk = rand_knots(rng, 1e-5, 1.0, 9)
    subs = [rand_knots(rng, 1.5, 4.0, 5), rand_knots(rng, 4.0, 90.0, 7)]
    vals = [rng.normal(size=(len(xk), len(q), 1)) for q in subs]
    vals[1][:, 0, :] = vals[0][:, -1, :]   # the same values on both copies of the threshold knot: f itself is continuous there
    g = oracle.OraclePdfGrid.from_spec(make_spec(xk, subs, [21], values=vals))
    e = 1e-6

    def slopes_x(xknot, q2):   # d f / d ln x just left and just right of the knot
        pts = np.array([xknot * np.exp(-e), xknot, xknot * np.exp(e)])
        f = g.xfxq2([21], pts, np.full(3, q2))[0]
        return (f[1] - f[0]) / e, (f[2] - f[1]) / e

    def slopes_q(x, q2knot):
        pts = np.array([q2knot * np.exp(-e), q2knot, q2knot * np.exp(e)])
        f = g.xfxq2([21], np.full(3, x), pts)[0]
        return (f[1] - f[0]) / e, (f[2] - f[1]) / e

    for q in (subs[0][1] ** 2 * 1.3, subs[1][3] ** 2 * 1.1):
        for xn in xk[1:-1]:
            l, r = slopes_x(xn, q)
            assert abs(l - r) < 2e-4 * max(1.0, abs(l)), (xn, l, r)
    jumps = []
    for x in (xk[2] * 1.2, xk[6] * 1.05):
        for s, qs in enumerate(subs):
            for qn in qs[1:-1]:
                l, r = slopes_q(x, qn ** 2)
                assert abs(l - r) < 2e-4 * max(1.0, abs(l)), (x, qn, l, r)
        l, r = slopes_q(x, subs[1][0] ** 2)   # the threshold: last knot of sub-grid 0 = first of sub-grid 1
        assert abs(l) < 1e3 and abs(r) < 1e3   # no jump of the value (that would be a slope ~ 1/e)
        jumps.append(abs(l - r))
    assert max(jumps) > 1e-2  # random values: the one-sided slopes of two independent sub-grids differ
