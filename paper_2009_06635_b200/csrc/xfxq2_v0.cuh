// xfxq2_v0.cuh -- the read-only-cache evaluation of one point (readings O3-O5): binary search on the
// raw knots, 64-byte interval records and the [iq][ix][kpad] value table through the read-only path.
// Used by k_xfxq2_v0 (xfxq2_kernels.cu: grids the shared-memory path does not take) and by the
// general kernel of pdf_lumi_events (lumi_kernels.cu: events with a point outside the grid).
#pragma once
#include "pdfb_internal.cuh"

struct ReqCols { int n; int col[PDFB_MAX_PIDS]; };

// largest m in [0, M-2] with k[m] <= v (0 if none): comparisons on raw values (reading Q5)
__device__ __forceinline__ int find_interval(const double *__restrict__ k, int M, double v)
{
    int lo = 0, hi = M - 1;  // invariant: answer in [lo, hi)
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (__ldg(k + mid) <= v) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ IntervalRec load_rec(const IntervalRec *p)
{
    const double2 *q = reinterpret_cast<const double2 *>(p);
    double2 a = __ldg(q), b = __ldg(q + 1), c = __ldg(q + 2), d = __ldg(q + 3);
    IntervalRec r = {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
    return r;
}

// O4 -- continuation E(z; zL, zH, yL, yH) with r = (z - zL)/(zH - zL) precomputed
__device__ __forceinline__ double continuation(double r, double yL, double yH)
{
    if (yL > 1e-3 && yH > 1e-3) {
        double lL = log(yL);
        return exp(fma(r, log(yH) - lL, lL));
    }
    return fma(r, yH - yL, yL);
}

// A "u-set" / "v-set": base knot index of a 4-wide stencil (already clamped so that all four
// indices are in range) and its weights.  Weights of knots that do not exist are exactly 0.
struct Set4 { int base; double w[4]; };

__device__ __forceinline__ Set4 make_set(int m, int M, const double w[4])
{
    // stencil knots m-1..m+2; shift the window into [0, M-1] keeping weights aligned
    Set4 s;
    int base = m - 1;
    int shift = 0;
    if (base < 0) shift = -base;               // m == 0: knot -1 has weight 0
    if (base + 3 > M - 1) shift = (M - 1) - (base + 3);  // m == M-2: knot M has weight 0
    if (M < 4) {                               // tiny arrays: place explicitly
        s.base = 0;
        for (int a = 0; a < 4; a++) s.w[a] = 0.0;
        for (int a = 0; a < 4; a++) { int k = m - 1 + a; if (k >= 0 && k < M) s.w[k] = w[a]; }
        return s;
    }
    s.base = base + shift;
    for (int a = 0; a < 4; a++) { int src = a + shift; s.w[a] = (src >= 0 && src < 4) ? w[src] : 0.0; }
    return s;
}

__device__ __forceinline__ double contract(const double *__restrict__ val, int kpad, int nx, int voff,
                                           const Set4 &us, const Set4 &vs, int nq, int col)
{
    double acc = 0.0;
#pragma unroll
    for (int b = 0; b < 4; b++) {
        int jq = min(vs.base + b, nq - 1);
        double row = 0.0;
#pragma unroll
        for (int a = 0; a < 4; a++) {
            int ix = min(us.base + a, nx - 1);
            row = fma(us.w[a], __ldg(val + ((long long)(voff + jq * nx + ix)) * kpad + col), row);
        }
        acc = fma(vs.w[b], row, acc);
    }
    return acc;
}


// One point, all requested columns, any region (readings O3-O5).  Returns false where no value is
// defined (x > x_max, x <= 0, Q^2 <= 0, NaN, Inf): res[] is then NaN.  `val` = the member's table.
__device__ __forceinline__ bool xf_point_v0(const GridDev &g, const double *__restrict__ val, const ReqCols &rc,
                                            double xv, double qv, double *res)
{
    if (!(xv > 0.0) || !(qv > 0.0) || !(xv <= g.x_max) || isinf(qv)) {
        for (int r = 0; r < rc.n; r++) res[r] = __longlong_as_double(0x7ff8000000000000LL);
        return false;
    }
    const bool low_x = xv < g.x_min, high_q = qv > g.q2_max, low_q = qv < g.q2_min;

    // ---- sub-grid of the point (O3 step 1; the Q^2 rules probe the last / the first sub-grid)
    int s = 0;
    if (high_q) s = g.n_sub - 1;
    else if (!low_q)
        for (int r = 1; r < g.n_sub; r++) if (g.q2_lo[r] <= qv) s = r;
    const int nq = g.q_off[s + 1] - g.q_off[s];
    // its x knots: one array for all sub-grids, or its own (pdf_grid_load_xs)
    const int xo = g.xs_per_sub ? g.x_off[s] : 0, nxs = g.xs_per_sub ? g.x_off[s + 1] - g.x_off[s] : g.nx;

    // ---- u direction: one set (in range) or the two one-hot sets of knots 0 and 1 (rule A)
    Set4 u1, u2;
    double rA = 0.0;
    if (!low_x) {
        int i = find_interval(g.xk + xo, nxs, xv);
        IntervalRec r = load_rec(g.xrec + xo + i);
        double w[4];
        weights4(r, (xv == g.x_max) ? 1.0 : (pdfb_ln(xv) - r.z0) * r.inv_dz, w);  // the last knot: t = 1 exactly (xfxq2_smem.cuh, t_coord)
        u1 = make_set(i, nxs, w);
    } else {
        rA = (pdfb_ln(xv) - g.U0) * (g.xs_per_sub ? g.inv_dU01s[s] : g.inv_dU01);
        u1.base = 0; u1.w[0] = 1.0; u1.w[1] = u1.w[2] = u1.w[3] = 0.0;
        u2.base = 0; u2.w[1] = 1.0; u2.w[0] = u2.w[2] = u2.w[3] = 0.0;
    }
    // ---- v direction: one set (in range), or two sets (rules B, C)
    Set4 v1, v2;
    double rB = 0.0;
    if (high_q) {  // probes at the last two Q^2 knots of the last sub-grid
        rB = (pdfb_ln(qv) - g.Va) * g.inv_dVab;
        int base = max(nq - 4, 0), ia = nq - 2 - base, ib = nq - 1 - base;
        v1.base = v2.base = base;
        for (int b = 0; b < 4; b++) { v1.w[b] = (b == ia) ? 1.0 : 0.0; v2.w[b] = (b == ib) ? 1.0 : 0.0; }
    } else if (low_q) {  // probes at q_min (knot 0 of sub-grid 0) and at 1.01 q_min
        v1.base = 0; v1.w[0] = 1.0; v1.w[1] = v1.w[2] = v1.w[3] = 0.0;
        v2 = make_set(g.jC, nq, g.wvC);
    } else {
        int j = find_interval(g.q2k + g.q_off[s], nq, qv);
        IntervalRec r = load_rec(g.qrec + g.q_off[s] + j);
        double w[4];
        weights4(r, (qv == g.q2_max) ? 1.0 : (pdfb_ln(qv) - r.z0) * r.inv_dz, w);
        v1 = make_set(j, nq, w);
    }
    const int voff = g.v_off[s];
    const bool two_v = high_q || low_q;
    const double rho = qv / g.q2_min;

    for (int r = 0; r < rc.n; r++) {
        int col = rc.col[r];
        double y1, y2 = 0.0;
        if (!low_x) {
            y1 = contract(val, g.kpad, nxs, voff, u1, v1, nq, col);
            if (two_v) y2 = contract(val, g.kpad, nxs, voff, u1, v2, nq, col);
        } else {  // rule A applied to each v probe
            y1 = continuation(rA, contract(val, g.kpad, nxs, voff, u1, v1, nq, col),
                              contract(val, g.kpad, nxs, voff, u2, v1, nq, col));
            if (two_v)
                y2 = continuation(rA, contract(val, g.kpad, nxs, voff, u1, v2, nq, col),
                                  contract(val, g.kpad, nxs, voff, u2, v2, nq, col));
        }
        double out = y1;
        if (high_q) {
            out = continuation(rB, y1, y2);
        } else if (low_q) {  // rule C: y0 * rho^(gamma*rho + 1 - rho)
            double gamma = 1.0;  // |y0| < 1e-5: y0 * rho (reading Q9)
            if (fabs(y1) >= 1e-5) gamma = fmax(-2.5, (y2 - y1) / y1 / 0.01);
            out = y1 * pow(rho, fma(gamma, rho, 1.0 - rho));
        }
        res[r] = out;
    }
    return true;
}
