// xfxq2_smem.cuh -- device code shared by the shared-memory path of pdf_xfxq2 (xfxq2_smem.cu: the
// kernel and its in-range loop; xfxq2_slow.cuh: the out-of-grid classes).  Layout of the staged
// slice, the conflict-free rotated gather and the LUT search are described in xfxq2_smem.cu.
#pragma once
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

// PDFB_CHECKED (build.py: PDFB_BUILD_FLAGS=-DPDFB_CHECKED): every shared-memory gather address is checked
// against the dynamic shared-memory window of the CTA, and the kernels poison the window with NaN
// before staging -- a read of anything that was not staged, even with weight 0, then shows up as a
// NaN output.  (compute-sanitizer is closed on the pool this was developed on; profiles/r2_sanitizer.md.)
#ifdef PDFB_CHECKED
#include <cassert>
__device__ __forceinline__ void pdfb_check_smem(uint32_t addr, uint32_t bytes)
{
    extern __shared__ __align__(128) unsigned char pdfb_dyn_smem[];  // every extern array is the dynamic window
    uint32_t size;
    asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(size));
    const uint32_t lo = (uint32_t)__cvta_generic_to_shared(pdfb_dyn_smem);
    assert(addr % bytes == 0 && addr >= lo && addr + bytes <= lo + size);
}
#define PDFB_ASSERT(c) assert(c)
#else
#define PDFB_ASSERT(c)
#endif

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
#ifdef PDFB_CHECKED
    pdfb_check_smem(addr, 16);
#endif
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ int2 lds64i(uint32_t addr)
{
#ifdef PDFB_CHECKED
    pdfb_check_smem(addr, 8);
#endif
    int2 v;
    asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
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

// The LAST knot of an axis (x = x_max, Q^2 = q2_max) starts a phantom interval of its own: its record is
// K1's pad entry {z_last, 1/dz = 0, 0, 0}, so t = 0 and the weights are (0, 1, 0, 0) EXACTLY -- the knot
// reproduces its table value bit for bit, like every other knot (which is the lower knot of its own
// interval), at no cost in the loop.  (As the upper end of the last real interval it would get
// t = (z1 - z0) * (1 / dz), which can round to 1 - 2^-53.)  Its stencil reaches two rows / two knots past
// the table with weight exactly 0: finite data lies there (pdfb_internal.cuh, "post").
__device__ __forceinline__ int locate_x(const GridDev &g, const SmemViews &sv, double xv, double u)
{
    return locate(sv.lutx, sv.xk, g.nx - 1, xv, u, g.lutx_u0, g.lutx_inv_h);
}

// Interval of Q^2 as an index into the CONCATENATED knot list.  A threshold is stored twice (last
// knot of the lower sub-grid, first of the upper), so a point on it lands on the upper copy
// (reading Q2) and the lower copy never starts an interval; Q^2 = q2_max lands on the last knot's
// phantom interval (above).  Interval records and table rows use the same index.
__device__ __forceinline__ int locate_q(const GridDev &g, const SmemViews &sv, double qv, double v)
{
    return locate(sv.lutq, sv.q2k, g.nq_tot - 1, qv, v, g.lutq_v0, g.lutq_inv_h);
}

template <int W> struct YW { double v[W]; };  // one point's W columns, in column order

// Kernel variants (compile-time): MODE = Q_IS_Q | OUT << 1.
//   Q_IS_Q  the scale array holds Q in GeV (pdf_xfxq), squared once on load
//   OUT     0: fp64, flavour-major out[r * stride + p]              (pdf_xfxq2, the contract layout)
//           1: fp64, point-major   out[p * n_req + r]               (pdf_xfxq2_pm)
//           2: fp32, flavour-major ((float *)out)[r * stride + p]   (pdf_xfxq2_f32: fp64 arithmetic, one rounding at the store)
#define PDFB_OUT_FM64 0
#define PDFB_OUT_PM64 1
#define PDFB_OUT_FM32 2

template <int OUT>
__device__ __forceinline__ void store_one(double *__restrict__ out, long long out_stride, int n_req, long long p, int r, double v)
{
    if (OUT == PDFB_OUT_FM64) __stcs(out + r * out_stride + p, v);
    else if (OUT == PDFB_OUT_PM64) __stcs(out + p * n_req + r, v);
    else __stcs(reinterpret_cast<float *>(out) + r * out_stride + p, (float)v);
}

// one point's W columns to their output rows (row < 0: column not requested)
template <int W, int OUT>
__device__ __forceinline__ void store_cols(double *__restrict__ out, long long out_stride, int n_req, long long p,
                                           const int row[W], const double v[W])
{
    if (row[0] >= 0) store_one<OUT>(out, out_stride, n_req, p, row[0], v[0]);
    if (row[1] >= 0) store_one<OUT>(out, out_stride, n_req, p, row[1], v[1]);
    if (W == 4) {
        if (row[W - 2] >= 0) store_one<OUT>(out, out_stride, n_req, p, row[W - 2], v[W - 2]);
        if (row[W - 1] >= 0) store_one<OUT>(out, out_stride, n_req, p, row[W - 1], v[W - 1]);
    }
}

// the scale of a point: Q^2, or Q in GeV squared once on load (a non-positive Q is invalid, like Q^2 <= 0)
template <bool Q_IS_Q>
__device__ __forceinline__ double load_scale(const double *p)
{
    const double q = __ldg(p);
    return Q_IS_Q ? ((q > 0.0) ? q * q : -1.0) : q;
}

