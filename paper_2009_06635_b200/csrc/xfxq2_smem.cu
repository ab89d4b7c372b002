// xfxq2_smem.cu -- K2/K3, the shared-memory path of pdf_xfxq2 (readings O3-O5).
//
// Why it looks the way it does ("Kernel design"): per point and flavour the method
// gathers a 4x4 value stencil -- 1408 B of table per point at 11 flavours against 104 B of HBM
// traffic -- and the points of a warp almost never share a cell.  The gather is what bounds the
// kernel, so it is fed from shared memory at full crossbar width, with no bank conflict:
//   * the value table is split into FLAVOUR GROUPS of 4 columns; one group's slice
//     [iq][ix4][4] (32 B per knot, iq over the concatenated Q^2 knots) fits shared memory and is
//     staged once per CTA by TMA bulk copies.  Each persistent CTA serves one group for all
//     points of its tiles, so it writes whole flavour rows with coalesced stores and no point
//     ever has to be re-ordered;
//   * the 4x4 stencil is always read as 4 consecutive rows x 4 consecutive knots, rows i-1..i+2 of
//     the concatenated table.  In an edge interval the stencil reaches one row / one knot outside
//     the knot array or the sub-grid; that knot carries weight exactly 0 (one-sided derivative
//     rule, reading O2), so whatever finite number sits there contributes nothing: a neighbouring
//     sub-grid's row, the next row's first knot, or the interval records that bracket the slice in
//     shared memory.  Rows are a uniform stride apart, so the 32 loads of a point use 8 per-lane
//     addresses + 3 uniform offsets (LDS [R+UR]) and no address arithmetic;
//   * one window row (4 knots x 4 flavours) is 128 contiguous bytes = 8 chunks of 16 B that
//     cover all 8 bank groups.  Lane l reads them in the rotated order c = (s + l - 2*node0) & 7,
//     so at every step the 8 lanes of a quarter-warp hit 8 distinct bank groups whatever cells
//     their points fell in: 32 conflict-free LDS.128 per point and group, 4 wavefronts each;
//   * the x weights are rotated the same way (selects on the ALU pipe), so no data is moved back.
// Knot location uses a uniform-in-log lookup table corrected by comparisons on the raw knots
// (the result is defined by the comparisons, reading Q5).
#include <cstdlib>

#include "pdfb_internal.cuh"

struct PassList {
    int n;
    int group[PDFB_MAX_PIDS];
    int row[PDFB_MAX_PIDS][4];  // output row of each of the group's 4 columns, -1 = not requested
};

#ifndef NT_SMEM
#define NT_SMEM 512   // threads per CTA (one CTA per SM: the slice fills shared memory)
#endif
#ifndef PPT_SMEM
#define PPT_SMEM 1    // points per thread and tile
#endif

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

// The continuation rules run on a few percent of the points at most but carry the fp64 log / exp /
// pow bodies: they are kept OUT of line (one copy each) so that the kernel stays within the
// instruction cache when warps alternate between the fast path and the out-of-grid lists
// (inlined they made the kernel 112 KB and a 30 % out-of-grid mix 3x slower than its parts).
__device__ __noinline__ double cont_e(double r, double yL, double yH)  // reading O4
{
    if (yL > 1e-3 && yH > 1e-3) {
        double lL = log(yL);
        return exp(fma(r, log(yH) - lL, lL));
    }
    return fma(r, yH - yL, yL);
}

// the coordinate logarithm of the out-of-grid path: pdfb_ln, one copy (code size, see cont_e)
__device__ __noinline__ double ln_slow(double a) { return pdfb_ln(a); }

// rule C (reading O5): y0 * rho^(gamma*rho + 1 - rho), gamma from the probe at 1.01 q_min;
// |y0| < 1e-5: gamma = 1, i.e. y0 * rho (reading Q9)
__device__ __noinline__ double rule_c(double y0, double y1, double rho)
{
    double gamma = 1.0;
    if (fabs(y0) >= 1e-5) gamma = fmax(-2.5, (y1 - y0) / y0 / 0.01);
    return y0 * pow(rho, fma(gamma, rho, 1.0 - rho));
}

// The four 1-D weights of knots m-1..m+2 from the 32-byte interval record.  aLm == 0 marks the
// first interval of the knot array (knot m-1 does not exist, weight exactly 0), aHp == 0 the last.
__device__ __forceinline__ void weights_rec32(const IntervalRec32 &r, double t, double w[4])
{
    // exact zero tests on the high words (the records hold +0.0 there), off the FP64 pipe
    const bool first = (__double2hiint(r.aLm) << 1) == 0, last = (__double2hiint(r.aHp) << 1) == 0;
    double t2 = t * t, t3 = t2 * t;
    double h01 = 3.0 * t2 - 2.0 * t3;
    double h00 = 1.0 - h01;
    double h11 = t3 - t2;
    double h10 = h11 - t2 + t;
    double aL1 = first ? 1.0 : 0.5, aH0 = last ? -1.0 : -0.5;
    double aL0 = -(r.aLm + aL1), aH1 = -(aH0 + r.aHp);
    w[0] = h10 * r.aLm;
    w[1] = fma(h11, aH0, fma(h10, aL0, h00));
    w[2] = fma(h11, aH1, fma(h10, aL1, h01));
    w[3] = h11 * r.aHp;
}

// o[k] = w[(k + r) & 3]
__device__ __forceinline__ void rot4(const double w[4], int r, double o[4])
{
    double a[4];
#pragma unroll
    for (int k = 0; k < 4; k++) a[k] = (r & 1) ? w[(k + 1) & 3] : w[k];
#pragma unroll
    for (int k = 0; k < 4; k++) o[k] = (r & 2) ? a[(k + 2) & 3] : a[k];
}

// The x side of a point's stencil.  The 128-byte run of knots node0..node0+3 (node0 = i-1, 4
// columns each) holds chunk c = 2*(knot - node0) + (column pair).  Lane l reads, at step s,
//   c(s) = ((s + rot) & 7) ^ (l & 1),   rot = ((l & 6) - 2*node0) & 7   (even),
// which puts the 8 lanes of a quarter-warp on 8 distinct bank groups at every step.  Steps 2k and
// 2k+1 both belong to knot (k + rot/2) & 3, so one rotated weight W[k] serves both; even steps
// deliver column pair (l & 1), odd steps the other pair (swapped back before the store).
struct Win { uint32_t a[8]; double W[4]; };

// row0 = shared address of stencil row 0 (table row gi-1); wu = x weights of knots node0..node0+3
__device__ __forceinline__ void make_win(Win &u, uint32_t row0, int node0, const double wu[4], int lane8)
{
    const int rot2 = ((lane8 >> 1) - node0) & 3;
    const uint32_t base = row0 + (uint32_t)(node0 * 32) + ((uint32_t)(lane8 & 1) << 4);
#pragma unroll
    for (int k = 0; k < 4; k++) {
        u.a[2 * k] = base + ((uint32_t)((k + rot2) & 3) << 5);
        u.a[2 * k + 1] = u.a[2 * k] ^ 16u;
    }
    rot4(wu, rot2, u.W);
}

// sum_b vw[b] * sum_k W[k] * V[window row b][window knot][cols] -> E = column pair (lane & 1), O = the other
__device__ __forceinline__ void gather4(const Win &u, const double vw[4], uint32_t rb1, uint32_t rb2, uint32_t rb3,
                                        double2 &yE, double2 &yO)
{
    yE = make_double2(0.0, 0.0); yO = make_double2(0.0, 0.0);
#pragma unroll
    for (int b = 0; b < 4; b++) {
        const uint32_t ro = (b == 0) ? 0u : (b == 1) ? rb1 : (b == 2) ? rb2 : rb3;
        double2 c[8];
#pragma unroll
        for (int s = 0; s < 8; s++) c[s] = lds128(u.a[s] + ro);
        double2 E, O;
        E.x = u.W[0] * c[0].x; E.y = u.W[0] * c[0].y;
        O.x = u.W[0] * c[1].x; O.y = u.W[0] * c[1].y;
#pragma unroll
        for (int k = 1; k < 4; k++) {
            E.x = fma(u.W[k], c[2 * k].x, E.x); E.y = fma(u.W[k], c[2 * k].y, E.y);
            O.x = fma(u.W[k], c[2 * k + 1].x, O.x); O.y = fma(u.W[k], c[2 * k + 1].y, O.y);
        }
        yE.x = fma(vw[b], E.x, yE.x); yE.y = fma(vw[b], E.y, yE.y);
        yO.x = fma(vw[b], O.x, yO.x); yO.y = fma(vw[b], O.y, yO.y);
    }
}

// ---- 2-column slices (16 B per knot).  A 4-knot run is 64 bytes = 4 bank groups; the row length is
// 64 (mod 128) bytes, so the same run one row further down covers the other 4.  A ROW PAIR is read as
// one virtual run of 8 chunks: chunk v < 4 = (upper row, knot v), v >= 4 = (lower row, knot v - 4),
// bank group (g0 + v) & 7.  Lane l reads v(s) = (s + l - g0) & 7 at step s: the 8 lanes of a
// quarter-warp are on 8 distinct bank groups whatever their cells.  16 conflict-free LDS.128 per
// point, each delivering both columns of one knot (no column-pair parity here).
__device__ __forceinline__ void stencil2(uint32_t row0, uint32_t RB, int node0, const double wu[4], const double vw[4],
                                         int lane8, double out[2])
{
    const uint32_t base = row0 + (uint32_t)(node0 * 16);
    const int rho = (lane8 - (int)(base >> 4)) & 7;  // g0 = bank group of the run's first chunk
    double Wr[4];
    rot4(wu, rho & 3, Wr);  // Wr[j] = weight of the knot read at steps s = j, j + 4
    uint32_t a[8];
    bool low[8];            // step s reads the lower row of the pair
#pragma unroll
    for (int s = 0; s < 8; s++) {
        const int v = (s + rho) & 7;
        low[s] = v >> 2;
        a[s] = base + (uint32_t)((v & 3) << 4) + (low[s] ? RB : 0u);
    }
    double y0 = 0.0, y1 = 0.0;
#pragma unroll
    for (int p = 0; p < 2; p++) {  // row pairs (0,1) and (2,3)
        double2 c[8];
#pragma unroll
        for (int s = 0; s < 8; s++) c[s] = lds128(a[s] + (p ? 2u * RB : 0u));
#pragma unroll
        for (int s = 0; s < 8; s++) {
            const double w = Wr[s & 3] * (low[s] ? vw[2 * p + 1] : vw[2 * p]);
            y0 = fma(w, c[s].x, y0); y1 = fma(w, c[s].y, y1);
        }
    }
    out[0] = y0; out[1] = y1;
}

// One stencil evaluation on a W-column slice: first stencil row `row` (table row gi-1), first knot
// node0 (= i-1); values come back in column order.
template <int W>
__device__ __forceinline__ void eval_stencil(uint32_t tab, uint32_t RB, uint32_t RB2, uint32_t RB3, int row, int node0,
                                             const double wu[4], const double vw[4], int lane8, double out[W])
{
    const uint32_t row0 = tab + (uint32_t)(row * (int)RB);
    if (W == 4) {
        Win w;
        make_win(w, row0, node0, wu, lane8);
        double2 E, O;
        gather4(w, vw, RB, RB2, RB3, E, O);
        const bool odd = lane8 & 1;  // E / O are the column pairs (lane & 1) / the other: back to column order
        out[0] = odd ? O.x : E.x; out[1] = odd ? O.y : E.y; out[W - 2] = odd ? E.x : O.x; out[W - 1] = odd ? E.y : O.y;
    } else {
        stencil2(row0, RB, node0, wu, vw, lane8, out);
    }
}

struct SmemViews {
    uint32_t tab, row_bytes, xrec, qrec;  // shared-space byte addresses
    const double *xk, *q2k;
    const unsigned short *lutx, *lutq;
};

// shared memory = [pre | slice | post] (pdfb_internal.cuh); the slice has W columns per knot
template <int W>
__device__ __forceinline__ SmemViews make_views(const GridDev &g, unsigned char *smem)
{
    SmemViews sv;
    const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(smem);
    sv.tab = s0 + (uint32_t)g.pre_bytes;
    sv.row_bytes = (W == 4) ? (uint32_t)g.nx4 * 32u : (uint32_t)g.nx2 * 16u;
    sv.xrec = s0 + (uint32_t)g.a_xrec;
    sv.qrec = sv.tab + (uint32_t)((W == 4 ? g.slice_bytes : g.slice2_bytes) + g.a_qrec);
    sv.xk = reinterpret_cast<const double *>(smem + g.a_xk);
    sv.q2k = reinterpret_cast<const double *>(smem + g.a_q2k);
    sv.lutx = reinterpret_cast<const unsigned short *>(smem + g.a_lutx);
    sv.lutq = reinterpret_cast<const unsigned short *>(smem + g.a_lutq);
    return sv;
}

// 32-byte interval record from its 128-byte line of 4 copies: lanes 2k and 2k+1 of a
// quarter-warp use copy k and read its two 16-byte halves in opposite order, so the 8 lanes
// touch 8 distinct bank groups at both steps whatever records they want.
__device__ __forceinline__ IntervalRec32 load_rec4(uint32_t line, int lane8)
{
    const uint32_t copy = line + (uint32_t)((lane8 >> 1) << 5);
    const uint32_t h = (uint32_t)(lane8 & 1) << 4;
    const double2 A = lds128(copy + h), B = lds128(copy + (h ^ 16u));
    IntervalRec32 r;
    r.z0 = h ? B.x : A.x; r.inv_dz = h ? B.y : A.y;
    r.aLm = h ? A.x : B.x; r.aHp = h ? A.y : B.y;
    return r;
}

// Interval search: LUT guess (pdfb_internal.cuh) + at most one comparison on the raw knots; bins
// holding several distinct knots take the comparison loop.  Returns the last m <= kmax with
// knots[m] <= val (the result is defined by the comparisons, reading Q5).
__device__ __forceinline__ int locate(const unsigned short *lut, const double *knots, int kmax, double val,
                                      double z, double z0, double inv_h)
{
    const int b = min(max((int)((z - z0) * inv_h), 0), PDFB_LUT_BINS - 1);
    const int e = lut[b], d = (e >> 1) & 3;
    int m = e >> 3;
    if (d) { if (knots[m + d] <= val) m += d; }
    if (e & 1)
        while (m < kmax && knots[m + 1] <= val) ++m;
    return m;
}

__device__ __forceinline__ int locate_x(const GridDev &g, const SmemViews &sv, double xv, double u)
{
    return locate(sv.lutx, sv.xk, g.nx - 2, xv, u, g.lutx_u0, g.lutx_inv_h);
}

// Interval of Q^2 as an index into the CONCATENATED knot list.  A threshold is stored twice (last
// knot of the lower sub-grid, first of the upper), so a point on it lands on the upper copy
// (reading Q2) and the lower copy never starts an interval; only Q^2 = q2_max needs the clamp.
// Interval records and table rows use the same index.
__device__ __forceinline__ int locate_q(const GridDev &g, const SmemViews &sv, double qv, double v)
{
    return min(locate(sv.lutq, sv.q2k, g.nq_tot - 1, qv, v, g.lutq_v0, g.lutq_inv_h), g.nq_tot - 2);
}

template <int W> struct YW { double v[W]; };  // one point's W columns, in column order

// one stencil evaluation of the out-of-grid path, out of line (see cont_e)
template <int W>
__device__ __noinline__ YW<W> probe(uint32_t tab, uint32_t RB, int row, int node0, const double *wu, const double *vw, int lane8)
{
    const double wu4[4] = {wu[0], wu[1], wu[2], wu[3]}, vw4[4] = {vw[0], vw[1], vw[2], vw[3]};
    YW<W> r;
    eval_stencil<W>(tab, RB, 2u * RB, 3u * RB, row, node0, wu4, vw4, lane8, r.v);
    return r;
}

// points outside the grid (readings O4/O5): up to 2 x-sets times 2 row sets
template <int W>
__device__ __noinline__ YW<W> slow_point(const GridDev *gp, unsigned char *smem, double xv, double qv, int lane8)
{
    const GridDev &g = *gp;
    const SmemViews sv = make_views<W>(g, smem);
    const uint32_t RB = sv.row_bytes;
    const bool low_x = xv < g.x_min, high_q = qv > g.q2_max, low_q = qv < g.q2_min;
    // ---- x: one weight set in range, else the two one-hot sets of knots 0 and 1 (rule A)
    double wu1[4] = {1.0, 0.0, 0.0, 0.0}, wu2[4] = {0.0, 1.0, 0.0, 0.0};  // knots 0..3
    int node0 = 0;
    double rA = 0.0;
    if (!low_x) {
        const double u = ln_slow(xv);
        const int i = locate_x(g, sv, xv, u);
        const IntervalRec32 r = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
        weights_rec32(r, (u - r.z0) * r.inv_dz, wu1);
        node0 = i - 1;
    } else {
        rA = (ln_slow(xv) - g.U0) * g.inv_dU01;
    }
    // ---- rows: one stencil in range, else two probes (rules B, C); row = table row of stencil row 0
    int row1, row2;
    double vw1[4], vw2[4];
    double rB = 0.0;
    if (high_q) {  // the last two Q^2 knots of the last sub-grid
        rB = (ln_slow(qv) - g.Va) * g.inv_dVab;
        row1 = row2 = g.nq_tot - 4;
        vw1[0] = vw1[1] = vw1[3] = 0.0; vw1[2] = 1.0;
        vw2[0] = vw2[1] = vw2[2] = 0.0; vw2[3] = 1.0;
    } else if (low_q) {  // q_min (row 0 of sub-grid 0) and 1.01 q_min (fixed interval and weights)
        row1 = 0;
        vw1[0] = 1.0; vw1[1] = vw1[2] = vw1[3] = 0.0;
        row2 = g.jC - 1;
#pragma unroll
        for (int b = 0; b < 4; b++) vw2[b] = g.wvC[b];
    } else {
        const double v = ln_slow(qv);
        const int gi = locate_q(g, sv, qv, v);
        const IntervalRec32 r = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
        weights_rec32(r, (v - r.z0) * r.inv_dz, vw1);
        row1 = row2 = gi - 1;
    }
    const bool two_v = high_q || low_q;
    YW<W> y1 = probe<W>(sv.tab, RB, row1, node0, wu1, vw1, lane8), y2 = y1;
    if (two_v) y2 = probe<W>(sv.tab, RB, row2, node0, wu1, vw2, lane8);
    if (low_x) {
        const YW<W> h1 = probe<W>(sv.tab, RB, row1, 0, wu2, vw1, lane8);
#pragma unroll
        for (int k = 0; k < W; k++) y1.v[k] = cont_e(rA, y1.v[k], h1.v[k]);
        if (two_v) {
            const YW<W> h2 = probe<W>(sv.tab, RB, row2, 0, wu2, vw2, lane8);
#pragma unroll
            for (int k = 0; k < W; k++) y2.v[k] = cont_e(rA, y2.v[k], h2.v[k]);
        }
    }
    const double rho = qv / g.q2_min;
#pragma unroll
    for (int k = 0; k < W; k++) {
        if (high_q) y1.v[k] = cont_e(rB, y1.v[k], y2.v[k]);
        else if (low_q) y1.v[k] = rule_c(y1.v[k], y2.v[k], rho);
    }
    return y1;
}

// one point's W columns to their output rows (row < 0: column not requested)
template <int W>
__device__ __forceinline__ void store_cols(double *__restrict__ out, long long out_stride, long long p,
                                           const int row[W], const double v[W])
{
    if (row[0] >= 0) __stcs(out + row[0] * out_stride + p, v[0]);
    if (row[1] >= 0) __stcs(out + row[1] * out_stride + p, v[1]);
    if (W == 4) {
        if (row[W - 2] >= 0) __stcs(out + row[W - 2] * out_stride + p, v[W - 2]);
        if (row[W - 1] >= 0) __stcs(out + row[W - 1] * out_stride + p, v[W - 1]);
    }
}

// the scale of a point: Q^2, or Q in GeV squared once on load (a non-positive Q is invalid, like Q^2 <= 0)
template <bool Q_IS_Q>
__device__ __forceinline__ double load_scale(const double *p)
{
    const double q = __ldg(p);
    return Q_IS_Q ? ((q > 0.0) ? q * q : -1.0) : q;
}

template <bool Q_IS_Q, int W>  // compile-time: a run-time flag costs 11 % (register pressure at the 128 cap)
__global__ void __launch_bounds__(NT_SMEM, 1)
k_xfxq2_smem(const __grid_constant__ GridDev g, const __grid_constant__ PassList pl, long long n,
             const double *__restrict__ x, const double *__restrict__ q2, double *__restrict__ out,
             long long out_stride, int member0, int n_req, int n_jobs)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) unsigned long long mbar;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // job = (member of the set, pass): blockIdx.x = seq * n_jobs + job; a job's CTAs share its tiles
    const int job = blockIdx.x % n_jobs, seq = blockIdx.x / n_jobs, nseq = gridDim.x / n_jobs;
    const int pass = job % pl.n, mem = job / pl.n;
    out += (long long)mem * n_req * out_stride;
    const uint32_t tab = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)g.pre_bytes;
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(&mbar);
    const int slice_bytes = (W == 4) ? g.slice_bytes : g.slice2_bytes;

    // ---- stage this CTA's flavour-group slice with TMA bulk copies; small tables by plain loads
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(slice_bytes) : "memory");
        const unsigned char *src = reinterpret_cast<const unsigned char *>(W == 4 ? g.valg : g.valg2) +
                                   ((size_t)(member0 + mem) * (W == 4 ? g.n_groups : g.n_groups2) + pl.group[pass]) * slice_bytes;
        for (int o = 0; o < slice_bytes; o += 32768) {
            int bytes = min(32768, slice_bytes - o);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(tab + o), "l"(src + o), "r"(bytes), "r"(mb) : "memory");
        }
    }
    {   // pre and post blocks around the slice (both multiples of 128 bytes)
        const int4 *src = reinterpret_cast<const int4 *>(g.aux);
        int4 *pre = reinterpret_cast<int4 *>(smem), *post = reinterpret_cast<int4 *>(smem + g.pre_bytes + slice_bytes);
        const int npre = g.pre_bytes / 16, npost = g.post_bytes / 16;
        for (int e = tid; e < npre; e += NT_SMEM) pre[e] = __ldg(src + e);
        for (int e = tid; e < npost; e += NT_SMEM) post[e] = __ldg(src + npre + e);
    }
    __syncthreads();
    {
        uint32_t done = 0;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(mb) : "memory");
    }
    const SmemViews sv = make_views<W>(g, smem);
    const int lane8 = tid & 7;
    const uint32_t RB = sv.row_bytes, rb2 = 2u * RB, rb3 = 3u * RB;
    const bool odd = lane8 & 1;
    const int row[4] = {pl.row[pass][0], pl.row[pass][1], pl.row[pass][2], pl.row[pass][3]};
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    // Out-of-grid points are not evaluated where they occur: each warp appends them to one list per
    // CLASS (0: x < x_min, 1: Q^2 > max, 2: Q^2 < min, 3 and 4: the corners 0+1, 0+2) and evaluates a
    // list when it holds a warp's worth, so that every slow_point call is class-uniform (no
    // divergence between the continuation rules) and runs on full lanes.  The lists live in a
    // global scratch slot owned by this SM (one CTA per SM at a time); counts are warp-uniform,
    // 6 bits per class in one register.
    unsigned cnts = 0;
    constexpr int TILE = NT_SMEM * PPT_SMEM;
    auto wlist = [&]() -> uint32_t * {
        uint32_t smid;
        asm("mov.u32 %0, %%smid;" : "=r"(smid));
        return g.slow_ws + ((size_t)(smid % PDFB_WS_SLOTS) * (NT_SMEM / 32) + warp) * (PDFB_SLOW_CLASSES * 32);
    };
    auto flush = [&](int cls, int count) {
        __syncwarp();
        if (lane < count) {
            const uint32_t e = __ldcg(wlist() + cls * 32 + lane);  // (iteration * PPT + k) << 5 | lane
            const uint32_t ik = e >> 5;
            const long long ps = ((long long)seq + (long long)(ik / PPT_SMEM) * nseq) * TILE + (ik % PPT_SMEM) * NT_SMEM +
                                 warp * 32 + (e & 31);
            const YW<W> r = slow_point<W>(&g, smem, __ldg(x + ps), load_scale<Q_IS_Q>(q2 + ps), lane8);
            store_cols<W>(out, out_stride, ps, row, r.v);
        }
        __syncwarp();
    };

    // software pipeline: the next tile's coordinates are in flight while this tile is evaluated
    long long tile = seq;
    double xv[PPT_SMEM], qv[PPT_SMEM];
#pragma unroll
    for (int k = 0; k < PPT_SMEM; k++) {
        const long long p = tile * TILE + k * NT_SMEM + tid;
        xv[k] = (p < n) ? __ldg(x + p) : 1.0; qv[k] = (p < n) ? load_scale<Q_IS_Q>(q2 + p) : 1.0;
    }
    for (uint32_t it = 0; tile * TILE < n; tile += nseq, ++it) {
        const long long p0 = tile * TILE + tid;
        double xn[PPT_SMEM], qn[PPT_SMEM];
        bool in_range[PPT_SMEM];
        bool any_in = false;
#pragma unroll
        for (int k = 0; k < PPT_SMEM; k++) {
            const long long pn = p0 + k * NT_SMEM + (long long)nseq * TILE;
            xn[k] = (pn < n) ? __ldg(x + pn) : 1.0; qn[k] = (pn < n) ? load_scale<Q_IS_Q>(q2 + pn) : 1.0;
            in_range[k] = (p0 + k * NT_SMEM < n) && xv[k] >= g.x_min && xv[k] <= g.x_max && qv[k] >= g.q2_min && qv[k] <= g.q2_max;
            any_in |= in_range[k];
        }
        if (any_in) {
            // ---- locate (LUT guess + exact comparisons where needed), weights, one gather per point.
            // A lane whose point is out of range computes a dummy in-range point and stores nothing.
#pragma unroll
            for (int k = 0; k < PPT_SMEM; k++) {
                const double xs = in_range[k] ? xv[k] : g.x_min, qs = in_range[k] ? qv[k] : g.q2_min;
                const double u = ln_pos(xs), v = ln_pos(qs);
                const int i = locate_x(g, sv, xs, u);
                const int gi = locate_q(g, sv, qs, v);
                const IntervalRec32 rx = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
                const IntervalRec32 rq = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
                double wu[4], vw[4], y[W];
                weights_rec32(rx, (u - rx.z0) * rx.inv_dz, wu);
                weights_rec32(rq, (v - rq.z0) * rq.inv_dz, vw);
                if (W == 4) {  // written out: the register allocation of this path is at the 128 cap
                    Win w;
                    make_win(w, tab + (uint32_t)((gi - 1) * (int)RB), i - 1, wu, lane8);
                    double2 E, O;
                    gather4(w, vw, RB, rb2, rb3, E, O);
                    y[0] = odd ? O.x : E.x; y[1] = odd ? O.y : E.y; y[W - 2] = odd ? E.x : O.x; y[W - 1] = odd ? E.y : O.y;
                } else {
                    eval_stencil<W>(tab, RB, rb2, rb3, gi - 1, i - 1, wu, vw, lane8, y);
                }
                if (in_range[k]) store_cols<W>(out, out_stride, p0 + k * NT_SMEM, row, y);
            }
        }
#pragma unroll
        for (int k = 0; k < PPT_SMEM; k++) {
            const long long p = p0 + k * NT_SMEM;
            const bool live = p < n;
            const bool invalid = live && !in_range[k] && (!(xv[k] > 0.0) || !(qv[k] > 0.0) || !(xv[k] <= g.x_max) || isinf(qv[k]));
            const bool slow = live && !in_range[k] && !invalid;
            const unsigned slow_mask = __ballot_sync(0xffffffffu, slow);
            if (invalid) {
                double nanv[W];
#pragma unroll
                for (int c = 0; c < W; c++) nanv[c] = qnan;
                store_cols<W>(out, out_stride, p, row, nanv);
                if (job == 0) atomicAdd(g.n_invalid, 1ULL);
            }
            if (slow_mask) {  // warp-uniform: append the out-of-grid points to their class lists
                const bool low_x = xv[k] < g.x_min, high_q = qv[k] > g.q2_max, low_q = qv[k] < g.q2_min;
                const int cls = low_x ? (high_q ? 3 : (low_q ? 4 : 0)) : (high_q ? 1 : 2);
                uint32_t *wl = wlist();
#pragma unroll
                for (int c = 0; c < PDFB_SLOW_CLASSES; c++) {
                    const unsigned m = __ballot_sync(0xffffffffu, slow && cls == c);
                    if (m) {
                        const int kc = __popc(m);
                        int cur = (cnts >> (6 * c)) & 63;
                        if (cur + kc > 32) { flush(c, cur); cur = 0; }
                        if (slow && cls == c)
                            __stcg(wl + c * 32 + cur + __popc(m & ((1u << lane) - 1u)), ((it * PPT_SMEM + k) << 5) | (uint32_t)lane);
                        cnts = (cnts & ~(63u << (6 * c))) | ((unsigned)(cur + kc) << (6 * c));
                    }
                }
            }
            xv[k] = xn[k]; qv[k] = qn[k];
        }
    }
#pragma unroll
    for (int c = 0; c < PDFB_SLOW_CLASSES; c++)
        if ((cnts >> (6 * c)) & 63) flush(c, (cnts >> (6 * c)) & 63);
}

static int smem_needed(const GridDev &d, int W) { return d.pre_bytes + (W == 4 ? d.slice_bytes : d.slice2_bytes) + d.post_bytes; }
static const int STATIC_SMEM = 256;  // >= the kernel's static shared memory (mbarrier)

// bit 0: the 4-column slices fit the device's shared memory, bit 1: the 2-column slices do
int pdfb_smem_eligible(const pdfb_grid *g)
{
    if (getenv("PDFB_FORCE_FALLBACK")) return 0;  // testing: force the read-only-cache path
    int dev_max = 0;
    if (cudaDeviceGetAttribute(&dev_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, g->device) != cudaSuccess) return 0;
    int ok = 0;
    if (smem_needed(g->d, 4) + STATIC_SMEM <= dev_max && !getenv("PDFB_NO_W4")) ok |= 1;  // (testing: 2-column path only)
    if (smem_needed(g->d, 2) + STATIC_SMEM <= dev_max) ok |= 2;
    if (!ok) return 0;
    // the attribute is per function, not per handle: raise it once to the device maximum
    static int attr_set_for = -1;
    if (attr_set_for != g->device) {
        const int lim = dev_max - STATIC_SMEM;
        if (cudaFuncSetAttribute(k_xfxq2_smem<false, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess ||
            cudaFuncSetAttribute(k_xfxq2_smem<true, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess ||
            cudaFuncSetAttribute(k_xfxq2_smem<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess ||
            cudaFuncSetAttribute(k_xfxq2_smem<true, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) != cudaSuccess) {
            cudaGetLastError();
            return 0;
        }
        attr_set_for = g->device;
    }
    return ok;
}

// passes of a request on W-column groups: one per (group, distinct use of its columns); a PID asked
// for twice gets an extra pass
static int build_passes(int W, int n_groups, int n_req, const int *cols, PassList &pl)
{
    pl.n = 0;
    bool used[PDFB_MAX_PIDS] = {false};
    for (int left = n_req; left > 0;) {
        for (int grp = 0; grp < n_groups && left > 0; grp++) {
            int row[4] = {-1, -1, -1, -1}, hit = 0;
            for (int r = 0; r < n_req; r++)
                if (!used[r] && cols[r] / W == grp && row[cols[r] % W] < 0) { row[cols[r] % W] = r; used[r] = true; hit++; }
            if (!hit) continue;
            if (pl.n >= PDFB_MAX_PIDS) return PDFB_ELIMIT;
            pl.group[pl.n] = grp;
            for (int k = 0; k < 4; k++) pl.row[pl.n][k] = row[k];
            pl.n++;
            left -= hit;
        }
    }
    return PDFB_OK;
}

int pdfb_launch_xfxq2_smem(const pdfb_grid *g, int n_req, const int *cols, long long n, const double *x,
                           const double *q2, double *out, long long out_stride, cudaStream_t st, int q_is_q,
                           int member0, int n_mem)
{
    // Width: a 4-column pass costs ~5.6 shared-memory wavefronts per point (4 gather + 1.6 setup and
    // I/O), a 2-column pass ~3.6; take the cheaper plan among the widths that fit shared memory.
    PassList pl4, pl2;
    pl4.n = pl2.n = 0;
    const int ok = g->d.smem_ok;
    int rc = PDFB_OK;
    if (ok & 1) rc = build_passes(4, g->d.n_groups, n_req, cols, pl4);
    if (!rc && (ok & 2)) rc = build_passes(2, g->d.n_groups2, n_req, cols, pl2);
    if (rc) return rc;
    const bool use2 = !(ok & 1) || ((ok & 2) && 3.6 * pl2.n < 5.6 * pl4.n);
    const PassList &pl = use2 ? pl2 : pl4;
    const int W = use2 ? 2 : 4;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device);
    // jobs = (member, pass).  Few jobs: the SMs are split between them and each CTA is persistent
    // over its share of the tiles.  More jobs than SMs: one CTA per job over all tiles, scheduled
    // by the hardware as SMs free up (one CTA per SM at a time: the slice fills shared memory).
    const long long n_jobs = (long long)pl.n * n_mem;
    if (n_jobs > 0x3fffffff) return PDFB_ELIMIT;
    int per_job = (int)(sms / n_jobs);
    if (per_job < 1) per_job = 1;
    long long tiles = (n + NT_SMEM * PPT_SMEM - 1) / (NT_SMEM * PPT_SMEM);
    if (per_job > tiles) per_job = (int)tiles;
    const unsigned grid = (unsigned)(per_job * n_jobs);
    const int smem = smem_needed(g->d, W);
#define PDFB_LAUNCH(Q, WW) k_xfxq2_smem<Q, WW><<<grid, NT_SMEM, smem, st>>>(g->d, pl, n, x, q2, out, out_stride, member0, n_req, (int)n_jobs)
    if (W == 4) { if (q_is_q) PDFB_LAUNCH(true, 4); else PDFB_LAUNCH(false, 4); }
    else        { if (q_is_q) PDFB_LAUNCH(true, 2); else PDFB_LAUNCH(false, 2); }
#undef PDFB_LAUNCH
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
