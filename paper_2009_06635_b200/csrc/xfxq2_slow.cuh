// xfxq2_slow.cuh -- points outside the grid (readings O4/O5), shared-memory path.
//
// The kernel (xfxq2_smem.cu) never evaluates such a point where it occurs.  Each warp appends the
// point's index to one list per continuation CLASS and evaluates whole batches of 32 entries, one
// class at a time, when a list of the CTA reaches the trigger length: every call below runs class-uniform on full
// warps, and all warps of the CTA run this code at about the same time instead of each alternating
// with the in-range loop on its own (which thrashed the instruction cache in round 1).
//
//   class 0  A   x < x_min, Q^2 in range      E(ln x; U0, U1, f(x0, Q^2), f(x1, Q^2))
//   class 1  B   Q^2 > q_max, x in range      E(ln Q^2; Va, Vb, f(x, qa), f(x, qb))
//   class 2  C   Q^2 < q_min, x in range      y0 rho^(gamma rho + 1 - rho), y0 = f(x, q_min), y1 = f(x, 1.01 q_min)
//   class 3  A+B, class 4  A+C                the Q^2 rule applied to values continued in x by rule A
//
// "Probes degenerate to one-hot weights": rule A needs knots 0 and 1 of the SAME
// 4-knot window, rule B the last two rows of the SAME 4-row window, so each takes ONE gather that
// keeps the two knots (rows) apart instead of two full stencil evaluations; the corners read eight
// warp-uniform table entries.
#pragma once
#include "xfxq2_smem.cuh"

// exp(x), |x| <= 700, ~1 ulp: x = k ln2 + r, |r| <= ln2 / 2, degree-13 Taylor polynomial (remainder
// r^14 / 14! < 5e-18), scaled through the exponent field.  (CUDA's exp costs about twice the
// instructions; the continuation rules below are bound by instruction issue.)
__device__ __forceinline__ double exp_small(double x)
{
    const double kf = rint(x * 1.4426950408889634074);
    double r = fma(-kf, c_ln[0], x);  // ln2_hi has 21 trailing zero bits: kf * ln2_hi is exact
    r = fma(-kf, c_ln[1], r);
    double p = 1.6059043836821613e-10;  // 1/13!
    p = fma(p, r, 2.08767569878681e-09);
    p = fma(p, r, 2.505210838544172e-08);
    p = fma(p, r, 2.755731922398589e-07);
    p = fma(p, r, 2.7557319223985893e-06);
    p = fma(p, r, 2.48015873015873e-05);
    p = fma(p, r, 1.984126984126984e-04);
    p = fma(p, r, 1.388888888888889e-03);
    p = fma(p, r, 8.333333333333333e-03);
    p = fma(p, r, 4.1666666666666664e-02);
    p = fma(p, r, 1.6666666666666666e-01);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    return __hiloint2double(__double2hiint(p) + ((int)kf << 20), __double2loint(p));
}
__device__ __noinline__ double exp_any(double x) { return (fabs(x) <= 700.0) ? exp_small(x) : exp(x); }

// reading O4, r = (z - zL)/(zH - zL) precomputed: exp(ln yL + r (ln yH - ln yL)) written as
// yL exp(r ln(yH / yL)) -- one division, one logarithm and one exponential per value instead of two
// logarithms and one exponential; the two forms differ by a few ulp times |r ln(yH/yL)|.
// Out of line: one copy of the bodies.
__device__ __noinline__ double cont_e(double r, double yL, double yH)
{
    if (yL > 1e-3 && yH > 1e-3) return yL * exp_any(r * ln_pos(yH / yL));
    return fma(r, yH - yL, yL);
}

// the coordinate logarithm of the out-of-grid classes: pdfb_ln, one copy
__device__ __noinline__ double ln_slow(double a) { return pdfb_ln(a); }

// rule C (reading O5): y0 * rho^(gamma*rho + 1 - rho) = y0 exp((gamma*rho + 1 - rho) ln rho), ln rho taken once
// per point; gamma from the probe at 1.01 q_min; |y0| < 1e-5: gamma = 1, i.e. y0 * rho (reading Q9)
__device__ __noinline__ double rule_c(double y0, double y1, double rho, double ln_rho)
{
    double gamma = 1.0;
    if (fabs(y0) >= 1e-5) gamma = fmax(-2.5, (y1 - y0) / y0 / 0.01);
    return y0 * exp_any(fma(gamma, rho, 1.0 - rho) * ln_rho);
}

// ---- x-contracted values of two consecutive table rows (rowA, rowA + RB), column order
template <int W>
__device__ __forceinline__ void rows_pair(uint32_t rowA, uint32_t RB, int node0, const double wu[4], int lane8,
                                          double ya[W], double yb[W])
{
    if (W == 4) {
        Win w;
        make_win(w, rowA, node0, wu, lane8);
        double2 E[2], O[2];
#pragma unroll
        for (int b = 0; b < 2; b++) {
            double2 c[8];
#pragma unroll
            for (int s = 0; s < 8; s++) c[s] = lds128(w.a[s] + (b ? RB : 0u));
            E[b].x = w.W[0] * c[0].x; E[b].y = w.W[0] * c[0].y;
            O[b].x = w.W[0] * c[1].x; O[b].y = w.W[0] * c[1].y;
#pragma unroll
            for (int k = 1; k < 4; k++) {
                E[b].x = fma(w.W[k], c[2 * k].x, E[b].x); E[b].y = fma(w.W[k], c[2 * k].y, E[b].y);
                O[b].x = fma(w.W[k], c[2 * k + 1].x, O[b].x); O[b].y = fma(w.W[k], c[2 * k + 1].y, O[b].y);
            }
        }
        const bool odd = lane8 & 1;
        ya[0] = odd ? O[0].x : E[0].x; ya[1] = odd ? O[0].y : E[0].y; ya[W - 2] = odd ? E[0].x : O[0].x; ya[W - 1] = odd ? E[0].y : O[0].y;
        yb[0] = odd ? O[1].x : E[1].x; yb[1] = odd ? O[1].y : E[1].y; yb[W - 2] = odd ? E[1].x : O[1].x; yb[W - 1] = odd ? E[1].y : O[1].y;
    } else {  // one row pair of the 2-column layout is one virtual 8-chunk run (stencil2)
        const uint32_t base = rowA + (uint32_t)(node0 * 16);
        const int rho = (lane8 - (int)(base >> 4)) & 7;
        double Wr[4];
        rot4(wu, rho & 3, Wr);
        double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
        double2 c[8];
#pragma unroll
        for (int s = 0; s < 8; s++) {
            const int v = (s + rho) & 7;
            c[s] = lds128(base + (uint32_t)((v & 3) << 4) + ((v >> 2) ? RB : 0u));
        }
#pragma unroll
        for (int s = 0; s < 8; s++) {
            const bool low = ((s + rho) & 7) >> 2;
            const double wa = low ? 0.0 : Wr[s & 3], wb = low ? Wr[s & 3] : 0.0;
            a0 = fma(wa, c[s].x, a0); a1 = fma(wa, c[s].y, a1);
            b0 = fma(wb, c[s].x, b0); b1 = fma(wb, c[s].y, b1);
        }
        ya[0] = a0; ya[1] = a1; yb[0] = b0; yb[1] = b1;
    }
}

// o = P[(j - r) & 3] for j = 0 and j = 1 (r in 0..3)
__device__ __forceinline__ void pick01(const double P[4], int r, double &o0, double &o1)
{
    const double a0 = (r & 1) ? P[3] : P[0], a1 = (r & 1) ? P[0] : P[1];  // (0 - r) & 3, (1 - r) & 3 for r = 0, 1
    const double b0 = (r & 1) ? P[1] : P[2], b1 = (r & 1) ? P[2] : P[3];  // ... for r = 2, 3
    o0 = (r & 2) ? b0 : a0; o1 = (r & 2) ? b1 : a1;
}

// ---- row-contracted values of x knots 0 and 1 (stencil rows row0 .. row0 + 3 RB), column order
template <int W>
__device__ __forceinline__ void knots_pair(uint32_t row0, uint32_t RB, const double vw[4], int lane8, double yL[W], double yH[W])
{
    if (W == 4) {
        const double dummy[4] = {0.0, 0.0, 0.0, 0.0};
        Win w;
        make_win(w, row0, 0, dummy, lane8);
        const int rot2 = (lane8 >> 1) & 3;  // steps 2k, 2k + 1 read knot (k + rot2) & 3
        double Ex[4], Ey[4], Ox[4], Oy[4];
#pragma unroll
        for (int k = 0; k < 4; k++) Ex[k] = Ey[k] = Ox[k] = Oy[k] = 0.0;
#pragma unroll
        for (int b = 0; b < 4; b++) {
            double2 c[8];
#pragma unroll
            for (int s = 0; s < 8; s++) c[s] = lds128(w.a[s] + (uint32_t)b * RB);
#pragma unroll
            for (int k = 0; k < 4; k++) {
                Ex[k] = fma(vw[b], c[2 * k].x, Ex[k]); Ey[k] = fma(vw[b], c[2 * k].y, Ey[k]);
                Ox[k] = fma(vw[b], c[2 * k + 1].x, Ox[k]); Oy[k] = fma(vw[b], c[2 * k + 1].y, Oy[k]);
            }
        }
        double eLx, eLy, oLx, oLy, eHx, eHy, oHx, oHy;
        pick01(Ex, rot2, eLx, eHx); pick01(Ey, rot2, eLy, eHy);
        pick01(Ox, rot2, oLx, oHx); pick01(Oy, rot2, oLy, oHy);
        const bool odd = lane8 & 1;
        yL[0] = odd ? oLx : eLx; yL[1] = odd ? oLy : eLy; yL[W - 2] = odd ? eLx : oLx; yL[W - 1] = odd ? eLy : oLy;
        yH[0] = odd ? oHx : eHx; yH[1] = odd ? oHy : eHy; yH[W - 2] = odd ? eHx : oHx; yH[W - 1] = odd ? eHy : oHy;
    } else {
        const int rho = (lane8 - (int)(row0 >> 4)) & 7;
        double Ax[4] = {0.0, 0.0, 0.0, 0.0}, Ay[4] = {0.0, 0.0, 0.0, 0.0};  // per step class j = s & 3: knot (j + rho) & 3
#pragma unroll
        for (int p = 0; p < 2; p++) {
            double2 c[8];
#pragma unroll
            for (int s = 0; s < 8; s++) {
                const int v = (s + rho) & 7;
                c[s] = lds128(row0 + (uint32_t)((v & 3) << 4) + ((v >> 2) ? RB : 0u) + (p ? 2u * RB : 0u));
            }
#pragma unroll
            for (int s = 0; s < 8; s++) {
                const double w = (((s + rho) & 7) >> 2) ? vw[2 * p + 1] : vw[2 * p];
                Ax[s & 3] = fma(w, c[s].x, Ax[s & 3]); Ay[s & 3] = fma(w, c[s].y, Ay[s & 3]);
            }
        }
        pick01(Ax, rho & 3, yL[0], yH[0]);
        pick01(Ay, rho & 3, yL[1], yH[1]);
    }
}

// one table entry (warp-uniform address in the corner classes): columns c, c + 1 of (row, knot)
template <int W>
__device__ __forceinline__ double2 entry2(uint32_t tab, uint32_t RB, int row, int knot, int c)
{
    return lds128(tab + (uint32_t)row * RB + (uint32_t)knot * (8u * W) + (uint32_t)c * 8u);
}

// ---- the x side of a point in range: window start and the four weights
__device__ __forceinline__ int x_side(const GridDev &g, const SmemViews &sv, double xv, int lane8, double wu[4])
{
    const double u = ln_slow(xv);
    const int i = locate_x(g, sv, xv, u);
    const IntervalRec32 r = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
    weights_rec32(r, (u - r.z0) * r.inv_dz, wu);
    return i - 1;
}

// class 0 (A)
template <int W>
__device__ __noinline__ YW<W> slow_A(const GridDev *gp, unsigned char *smem, double xv, double qv, int lane8)
{
    const GridDev &g = *gp;
    const SmemViews sv = make_views<W>(g, smem);
    const double v = ln_slow(qv);
    const int gi = locate_q(g, sv, qv, v);
    const IntervalRec32 r = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
    double vw[4], yL[W], yH[W];
    weights_rec32(r, (v - r.z0) * r.inv_dz, vw);
    knots_pair<W>(sv.tab + (uint32_t)((gi - 1) * (int)sv.row_bytes), sv.row_bytes, vw, lane8, yL, yH);
    const double rA = (ln_slow(xv) - g.U0) * g.inv_dU01;
    YW<W> y;
#pragma unroll
    for (int k = 0; k < W; k++) y.v[k] = cont_e(rA, yL[k], yH[k]);
    return y;
}

// class 1 (B): the last two Q^2 knots of the last sub-grid = the last two table rows
template <int W>
__device__ __noinline__ YW<W> slow_B(const GridDev *gp, unsigned char *smem, double xv, double qv, int lane8)
{
    const GridDev &g = *gp;
    const SmemViews sv = make_views<W>(g, smem);
    double wu[4], ya[W], yb[W];
    const int node0 = x_side(g, sv, xv, lane8, wu);
    rows_pair<W>(sv.tab + (uint32_t)(g.nq_tot - 2) * sv.row_bytes, sv.row_bytes, node0, wu, lane8, ya, yb);
    const double rB = (ln_slow(qv) - g.Va) * g.inv_dVab;
    YW<W> y;
#pragma unroll
    for (int k = 0; k < W; k++) y.v[k] = cont_e(rB, ya[k], yb[k]);
    return y;
}

// class 2 (C): q_min = row 0 of sub-grid 0; 1.01 q_min has a fixed interval jC and fixed weights wvC
template <int W>
__device__ __noinline__ YW<W> slow_C(const GridDev *gp, unsigned char *smem, double xv, double qv, int lane8)
{
    const GridDev &g = *gp;
    const SmemViews sv = make_views<W>(g, smem);
    const uint32_t RB = sv.row_bytes;
    double wu[4], y0[W], unused[W], y1[W];
    const int node0 = x_side(g, sv, xv, lane8, wu);
    rows_pair<W>(sv.tab, RB, node0, wu, lane8, y0, unused);
    const double wv[4] = {g.wvC[0], g.wvC[1], g.wvC[2], g.wvC[3]};
    eval_stencil<W>(sv.tab, RB, 2u * RB, 3u * RB, g.jC - 1, node0, wu, wv, lane8, y1);
    const double rho = qv / g.q2_min, ln_rho = ln_slow(rho);
    YW<W> y;
#pragma unroll
    for (int k = 0; k < W; k++) y.v[k] = rule_c(y0[k], y1[k], rho, ln_rho);
    return y;
}

// classes 3 (A+B) and 4 (A+C): knots 0 and 1 of fixed rows -- warp-uniform table entries
template <int W, bool HIGH_Q>
__device__ __noinline__ YW<W> slow_corner(const GridDev *gp, unsigned char *smem, double xv, double qv)
{
    const GridDev &g = *gp;
    const SmemViews sv = make_views<W>(g, smem);
    const uint32_t RB = sv.row_bytes;
    const double rA = (ln_slow(xv) - g.U0) * g.inv_dU01;
    const double rB = HIGH_Q ? (ln_slow(qv) - g.Va) * g.inv_dVab : 0.0;
    const double rho = qv / g.q2_min, ln_rho = HIGH_Q ? 0.0 : ln_slow(rho);
    YW<W> y;
#pragma unroll
    for (int c = 0; c < W; c += 2) {
        double2 p1[2], p2[2];  // probe 1 / probe 2 of the Q^2 rule at knot 0, knot 1
#pragma unroll
        for (int k = 0; k < 2; k++) {
            if (HIGH_Q) {
                p1[k] = entry2<W>(sv.tab, RB, g.nq_tot - 2, k, c);
                p2[k] = entry2<W>(sv.tab, RB, g.nq_tot - 1, k, c);
            } else {
                p1[k] = entry2<W>(sv.tab, RB, 0, k, c);
                double2 acc = make_double2(0.0, 0.0);
#pragma unroll
                for (int b = 0; b < 4; b++) {  // rows jC-1 .. jC+2; a row before the table has weight exactly 0 (finite data there)
                    const double2 e = lds128(sv.tab + (uint32_t)((g.jC - 1 + b) * (int)RB) + (uint32_t)k * (8u * W) + (uint32_t)c * 8u);
                    acc.x = fma(g.wvC[b], e.x, acc.x); acc.y = fma(g.wvC[b], e.y, acc.y);
                }
                p2[k] = acc;
            }
        }
        const double a1x = cont_e(rA, p1[0].x, p1[1].x), a1y = cont_e(rA, p1[0].y, p1[1].y);
        const double a2x = cont_e(rA, p2[0].x, p2[1].x), a2y = cont_e(rA, p2[0].y, p2[1].y);
        y.v[c] = HIGH_Q ? cont_e(rB, a1x, a2x) : rule_c(a1x, a2x, rho, ln_rho);
        y.v[c + 1] = HIGH_Q ? cont_e(rB, a1y, a2y) : rule_c(a1y, a2y, rho, ln_rho);
    }
    return y;
}

// `count` entries of one class list of this warp (a multiple of 32 except at the very end), 32 at a time.
template <int MODE, int W>
__device__ __noinline__ void flush_class(int cls, int count, const uint32_t *list, const GridDev *gp, unsigned char *smem,
                                         const double *__restrict__ x, const double *__restrict__ q2, double *__restrict__ out,
                                         long long out_stride, int n_req, const int *rowp)
{
    constexpr bool Q_IS_Q = MODE & 1;
    const int lane = threadIdx.x & 31, lane8 = threadIdx.x & 7;
    const int row[4] = {rowp[0], rowp[1], rowp[2], rowp[3]};
    for (int e = lane; e < count; e += 32) {
        const long long p = (long long)__ldcg(list + e);
        const double xv = __ldg(x + p), qv = load_scale<Q_IS_Q>(q2 + p);
        YW<W> r;
        switch (cls) {  // uniform over the warp
        case 0: r = slow_A<W>(gp, smem, xv, qv, lane8); break;
        case 1: r = slow_B<W>(gp, smem, xv, qv, lane8); break;
        case 2: r = slow_C<W>(gp, smem, xv, qv, lane8); break;
        case 3: r = slow_corner<W, true>(gp, smem, xv, qv); break;
        default: r = slow_corner<W, false>(gp, smem, xv, qv); break;
        }
        store_cols<W, (MODE >> 1)>(out, out_stride, n_req, p, row, r.v);
    }
}

// The full batches (final: all entries) of this warp's class lists; a remainder moves to the front.
template <int MODE, int W>
__device__ __noinline__ void flush_warp_lists(bool final, uint32_t *wl, unsigned char *cnt, unsigned char *req, const GridDev *gp,
                                              unsigned char *smem, const double *__restrict__ x, const double *__restrict__ q2,
                                              double *__restrict__ out, long long out_stride, int n_req, const int *rowp)
{
    const int lane = threadIdx.x & 31;
    __syncwarp();
    if (lane == 0) *req = 0;
#pragma unroll 1
    for (int c = 0; c < PDFB_SLOW_CLASSES; c++) {
        const int n = cnt[c];
        const int take = final ? n : (n & ~31);
        if (take == 0) continue;
        uint32_t *list = wl + c * PDFB_SLOW_LCAP;
        flush_class<MODE, W>(c, take, list, gp, smem, x, q2, out, out_stride, n_req, rowp);
        const int rem = n - take;  // < 32: moved to the front of the list
        uint32_t keep = 0;
        if (lane < rem) keep = __ldcg(list + take + lane);
        __syncwarp();
        if (lane < rem) __stcg(list + lane, keep);
        if (lane == 0) cnt[c] = (unsigned char)rem;
        __syncwarp();
    }
}

