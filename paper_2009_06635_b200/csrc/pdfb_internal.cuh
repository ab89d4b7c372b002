// pdfb_internal.cuh -- device-side data layout shared by the library's own translation units.
// (Nothing under oracle/ includes this file, and this file includes nothing from oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/pdfb200.h"

// One record per knot interval [z_m, z_{m+1}] of a 1-D knot array (x knots, or the Q^2 knots
// of one sub-grid).  Written once by the grid-setup kernel K1 (reading O2: finite-difference
// derivative rule).  With h00,h10,h01,h11 the cubic Hermite basis at
// t = (z - z0) * inv_dz, the interpolant on the interval is  sum_a w_a y_{m-1+a}  with
//   w_0 = h10*aLm,  w_1 = h00 + h10*aL0 + h11*aH0,  w_2 = h01 + h10*aL1 + h11*aH1,  w_3 = h11*aHp
// i.e. dz * (derivative at knot m)   = aLm*y_{m-1} + aL0*y_m + aL1*y_{m+1}
//      dz * (derivative at knot m+1) = aH0*y_m + aH1*y_{m+1} + aHp*y_{m+2}
// At the first (last) interval of the array aLm (aHp) is exactly 0 and the derivative is the
// one-sided slope.
struct __align__(16) IntervalRec {
    double z0;      // ln of the lower knot
    double inv_dz;  // 1 / (ln upper - ln lower)
    double aLm, aL0, aL1;
    double aH0, aH1, aHp;
};
static_assert(sizeof(IntervalRec) == 64, "IntervalRec must be 64 bytes");

// the four 1-D weights of knots m-1..m+2 at in-interval coordinate t (see IntervalRec)
__host__ __device__ __forceinline__ void weights4(const IntervalRec &r, double t, double w[4])
{
    double t2 = t * t, t3 = t2 * t;
    double h01 = 3.0 * t2 - 2.0 * t3;
    double h00 = 1.0 - h01;
    double h11 = t3 - t2;
    double h10 = h11 - t2 + t;
    w[0] = h10 * r.aLm;
    w[1] = fma(h11, r.aH0, fma(h10, r.aL0, h00));
    w[2] = fma(h11, r.aH1, fma(h10, r.aL1, h01));
    w[3] = h11 * r.aHp;
}

// ---------------------------------------------------------------------------------------------
// ln of a positive, finite, normal double.  Classic argument reduction m in [sqrt(1/2), sqrt(2)),
// s = f/(2+f), odd series in s, < 1 ulp; coefficients live in constant memory so that they are
// operands, not moves.  The reduction constant, the split of ln 2 and the minimax coefficients
// Lg1..Lg7 below are those of fdlibm's e_log.c, whose notice is reproduced as its licence asks:
//
//   ====================================================
//   Copyright (C) 1993 by Sun Microsystems, Inc. All rights reserved.
//
//   Developed at SunSoft, a Sun Microsystems, Inc. business.
//   Permission to use, copy, modify, and distribute this
//   software is freely granted, provided that this notice
//   is preserved.
//   ====================================================
//
// (the division of that routine is replaced here by a reciprocal seed + Newton steps + residual).
static __constant__ double c_ln[10] = {
    6.93147180369123816490e-01,  // ln2_hi
    1.90821492927058770002e-10,  // ln2_lo
    6.666666666666735130e-01,    // Lg1
    3.999999999940941908e-01,    // Lg2
    2.857142874366239149e-01,    // Lg3
    2.222219843214978396e-01,    // Lg4
    1.818357216161805012e-01,    // Lg5
    1.531383769920937332e-01,    // Lg6
    1.479819860511658591e-01,    // Lg7
    0.0};

__device__ __forceinline__ double ln_pos(double a)
{
    int hi = __double2hiint(a), lo = __double2loint(a);
    int k = (hi >> 20) - 1023;
    hi &= 0x000fffff;
    const int i = (hi + 0x95f64) & 0x100000;  // mantissa above sqrt(2): halve it
    k += i >> 20;
    const double m = __hiloint2double(hi | (i ^ 0x3ff00000), lo);
    const double f = m - 1.0;
    const double d = 2.0 + f;
    // s = f / d, correctly rounded in all but rare cases: reciprocal seed + Newton + residual
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    double s = f * r;
    s = fma(fma(-d, s, f), r, s);
    const double dk = (double)k;
    const double z = s * s, w = z * z;
    const double t1 = w * fma(w, fma(w, c_ln[7], c_ln[5]), c_ln[3]);
    const double t2 = z * fma(w, fma(w, fma(w, c_ln[8], c_ln[6]), c_ln[4]), c_ln[2]);
    const double R = t2 + t1;
    const double hfsq = 0.5 * f * f;
    return fma(dk, c_ln[0], -((hfsq - fma(s, hfsq + R, dk * c_ln[1])) - f));
}

// ln of any positive finite double (reading R-ln: every coordinate logarithm of the library --
// knots at load time, queries at run time -- goes through this one function, so a query that
// sits on a knot gets t = 0 exactly)
__device__ __forceinline__ double pdfb_ln(double a)
{
    return (a >= 2.2250738585072014e-308) ? ln_pos(a) : log(a);
}

// ---------------------------------------------------------------------------------------------
// ln of a positive normal double through a 64-entry table (alpha_s fast path, alphas_kernels.cu):
// a = 2^k m, m in [1, 2); c = 1 + (j + 1/2)/64 the centre of m's bin j (the top 6 mantissa bits);
// ln a = k ln2 + ln c + log1p(m/c - 1), |m/c - 1| < 2^-7, series to the 7th power (remainder < 2^-59).
// Absolute error a few 1e-16 + |k| ulp-level terms: ~1e-15 at |ln a| ~ 25.  alpha_s(t) moves by at
// most ~0.1 alpha per unit t = (ln Q^2 - Z_m)/dZ, so the 1e-12 rule needs |error of ln| < 1e-11 dZ:
// four orders of magnitude to spare on any sensible node list -- and less than half the instructions
// of ln_pos (no reciprocal).  The node logarithms of the fast path are taken with the same function,
// so a query on a node still gets t = 0 exactly.  Table entry = {1/c, ln c}, 8 copies per 128-byte
// line (a lane reads copy lane & 7: conflict-free).
#define PDFB_LNTAB_BYTES (64 * 128)
__device__ __forceinline__ int ln_tab_bin(double a) { return (__double2hiint(a) >> 14) & 63; }
__device__ __forceinline__ double ln_tab(double a, double2 e)
{
    const int hi = __double2hiint(a);
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, __double2loint(a));
    const double kf = (double)((hi >> 20) - 1023);
    const double r = fma(m, e.x, -1.0);
    double p = fma(r, 1.0 / 7.0, -1.0 / 6.0);
    p = fma(p, r, 0.2);
    p = fma(p, r, -0.25);
    p = fma(p, r, 1.0 / 3.0);
    p = fma(p, r, -0.5);
    p = fma(p * r, r, r);  // log1p(r)
    return fma(kf, c_ln[0], (e.y + fma(kf, c_ln[1], p)));
}

struct GridDev {
    int n_sub, nx, n_pid, nq_tot;
    int n_members;                     // member tables sharing these knots (pdf_set_load)
    long long val_mstride;             // doubles between two members in `val`
    int kpad;                          // doubles per knot in `val` (>= n_pid)
    int q_off[PDFB_MAX_SUBGRIDS + 1];  // knot offsets of the sub-grids
    int v_off[PDFB_MAX_SUBGRIDS];      // offset (in knots) of sub-grid s in `val`
    double q2_lo[PDFB_MAX_SUBGRIDS];   // first Q^2 knot of each sub-grid
    double x_min, x_max, q2_min, q2_max;
    // continuation (readings O4/O5)
    double U0, U1, inv_dU01;           // ln x_0, ln x_1, 1/(U1-U0)
    double Va, Vb, inv_dVab;           // ln of the last two Q^2 knots, 1/(Vb-Va)
    int jC;                            // interval of 1.01*q2_min in sub-grid 0
    double wvC[4];                     // its four v weights (fixed per grid), stencil order j-1..j+2
    // sub-grids with their own x-knot arrays (pdf_grid_load_xs; read-only-cache kernel only): sub-grid s owns
    // xk / xrec [x_off[s], x_off[s+1]); rule A continues from its first two knots: U0, inv_dU01s[s]
    int xs_per_sub;
    int x_off[PDFB_MAX_SUBGRIDS + 1];
    double inv_dU01s[PDFB_MAX_SUBGRIDS];
    const double *xk;                  // [nx] x knots
    const double *q2k;                 // [nq_tot] Q^2 knots
    const IntervalRec *xrec;           // [nx-1]
    const IntervalRec *qrec;           // [nq_tot]; entry q_off[s]+j = interval j of sub-grid s
    const double *val;                 // [member][s][iq][ix][kpad]: knot (s,ix,iq) at v_off[s]+iq*nx+ix
    unsigned long long *n_invalid;     // sticky counter
    int *row_range;                    // smem path: (PDFB_RR_SLOTS + PDFB_RR_CAP_SLOTS) x {first row, end row} staged by a small-batch call (xfxq2_smem.cu)
    uint32_t *slow_ws;                 // smem path: per SM and warp, PDFB_SLOW_CLASSES lists of out-of-grid point indices
    // ---- shared-memory path (xfxq2_smem.cu): flavour-group slices + a small aux block
    int smem_ok;                       // bit 0: the 4-column slices fit shared memory; bit 1: the 2-column ones
                                       // (0 if nx < 4 or a sub-grid has < 4 Q knots: read-only-cache kernel)
    int n_groups, nx4;                 // groups of 4 value columns; nx padded to a multiple of 4
    int slice_bytes;                   // one group's slice: nq_tot * nx4 * 32 B
    const double *valg;                // [member][group][s][iq][ix4][4]
    // 2-column slices: half the bytes per knot, for grids whose 4-column slice exceeds shared memory
    // and for requests of one or two flavours.  nx2 = 4 (mod 8), so that a row is 64 (mod 128) bytes
    // long and two consecutive rows of a 4-knot run cover all 8 bank groups (xfxq2_smem.cu)
    int n_groups2, nx2, slice2_bytes;
    const double *valg2;               // [member][group2][s][iq][nx2][2]
    const unsigned char *aux;          // [pre | post] blocks, copied verbatim around the slice
    int pre_bytes, post_bytes;         // shared memory = [pre | slice | post]
    int a_xk, a_q2k, a_lutx, a_lutq, a_xrec;  // byte offsets inside pre (a_xrec is its tail)
    int a_qrec;                        // byte offset inside post (its head)
    double lutx_u0, lutx_inv_h, lutq_v0, lutq_inv_h;
};
#ifndef PDFB_LUT_BINS
#define PDFB_LUT_BINS 512
#endif
#define PDFB_RR_SLOTS 64      // row-range slots of a handle: calls in flight on one handle that may use one each
#define PDFB_RR_CAP_SLOTS 64  // ... and as many again that only calls recorded by a stream capture take: a recorded call
                              // keeps its slot for every replay of its graph, so it must not sit in the live calls' ring
#define PDFB_SLOW_CLASSES 5   // x < x_min | Q^2 > max | Q^2 < min | the two corners
#define PDFB_WS_SLOTS 160     // >= %nsmid (148 on B200; checked at load): one scratch slot per SM
#ifndef PDFB_SLOW_TRIGGER
#define PDFB_SLOW_TRIGGER 192  // a list this long asks every warp of the CTA to evaluate its full batches
#endif
#define PDFB_SLOW_LCAP 256     // entries per warp and class list; 8-bit counters: TRIGGER - 1 + 32 + 31 <= 255
#define PDFB_WS_BYTES ((size_t)PDFB_WS_SLOTS * 16 * PDFB_SLOW_CLASSES * PDFB_SLOW_LCAP * 4)  // 16 warps per CTA
// Shared-memory image of the smem path: [pre | slice | post].
//   pre  = lutx, lutq, raw x knots, raw Q^2 knots, then xrec;   post = qrec, then zero padding.
// xrec/qrec = 128-byte lines holding 4 copies of the 32-byte IntervalRec32 of an interval (qrec is
// indexed by the concatenated Q^2 knot index).  The slice is bracketed by xrec and qrec ON PURPOSE:
// the 4x4 stencil of an edge interval reaches one row / one knot outside the table with weight
// exactly 0 (one-sided rule, reading O2), and what it reads there must be finite doubles.
// lut[b] = (m0 << 3) | (delta << 1) | multi, where m0 is the last knot at or left of the bin's
// left edge; if exactly one knot value lies inside the bin, delta = (index of its last copy) - m0
// and the interval is m0 + delta iff knots[m0 + delta] <= the raw coordinate, else m0; `multi`
// (several distinct knots in the bin) asks for the comparison loop.  A Q^2 threshold is stored
// twice in the concatenated list, so a point on it lands on the upper copy (reading Q2).

// 32-byte interval record of the shared-memory path: the remaining coefficients follow from
// "a derivative annihilates constants": aL1 = (aLm == 0 ? 1 : 1/2), aL0 = -(aLm + aL1),
// aH0 = (aHp == 0 ? -1 : -1/2), aH1 = -(aH0 + aHp).
struct __align__(16) IntervalRec32 { double z0, inv_dz, aLm, aHp; };

struct AlphasDev {
    int K, n_sub;
    int off[PDFB_MAX_SUBGRIDS + 1];
    double q2_lo[PDFB_MAX_SUBGRIDS];
    double q2_min, q2_max, a_first, a_last;
    const double *q2k;        // [K]
    const double *a;          // [K]
    const IntervalRec *rec;   // [K]
    // fast path (alphas_kernels.cu): per interval 3 lines of 128 B: {ln knot Z, d0} x 8, {d1, d2} x 8, d3 x 16,
    // so lane l reads copy (l & 7) of the first two (LDS.128) and copy (l & 15) of the third (LDS.64):
    // conflict-free whatever intervals the lanes want.  alpha_s = d0 + s(d1 + s(d2 + s d3)), s = ln Q^2 - Z.
    int fast_ok;
    const unsigned char *fast;  // [lines: K*384 B][ln table: PDFB_LNTAB_BYTES][q2k: K doubles][lut: PDFB_LUT_BINS u16]
    int fast_bytes, f_lntab, f_q2k, f_lut;
    double lut_v0, lut_inv_h;
};

// pdf_lumi_events (lumi_kernels.cu): shared-memory plan of the band kernel
struct LumiLayout {
    int R, R_alloc, CB, n_bands, ncell;
    int RB2;          // bytes per row of a 2-column slice
    int pair_stride;  // bytes between the bands of two pairs in shared memory (a multiple of 128)
    int l_band, l_qrec, l_list, total;
};

// Makes the handle's device current for the duration of a call and puts the caller's device back.
struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int device)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; ok = false; return; }
        if (prev != device) { if (cudaSetDevice(device) != cudaSuccess) ok = false; }
        else prev = -1;  // nothing to restore
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

struct pdfb_grid {
    int device;
    int sms;                  // multiprocessors of `device`
    std::atomic<unsigned> rr_next;  // next row-range slot (round robin)
    std::atomic<unsigned> rr_cap_next;  // next row-range slot of a call recorded by a stream capture
    LumiLayout lumi;          // band plan of pdf_lumi_events
    int lumi_npair;           // its kernel instance (column pairs staged per band); 0 = general kernel only
    GridDev d;
    int pids[PDFB_MAX_PIDS];
    void *blob;               // one device allocation holding all tables
    size_t blob_bytes;
    // staging for pdf_xfxq2_host
    void *stage;
    size_t stage_bytes;
    cudaStream_t streams[3];
    double setup_ms;
};

struct pdfb_alphas {
    int device;
    int sms;
    AlphasDev d;
    void *blob;
    void *stage;
    size_t stage_bytes;
    cudaStream_t streams[2];
};

// search LUT (capi.cu); encoding above
void pdfb_fill_lut(unsigned short *lut, const double *Z, const double *R, int nk, int kmax);

// launch accounting (capi.cu)
void pdfb_count_launch(int n);

// kernels' host launchers
// mode = Q_IS_Q | OUT << 1 (xfxq2_smem.cuh): bit 0: the scale array holds Q in GeV, squared once on load;
// OUT 0 / 1 / 2: fp64 flavour-major / fp64 point-major / fp32 flavour-major output
int pdfb_launch_xfxq2(const pdfb_grid *g, int n_req, const int *cols, long long n, const double *x,
                      const double *q2, double *out, long long out_stride, cudaStream_t st, int mode = 0,
                      int member0 = 0, int n_mem = 1);
int pdfb_launch_alphas(const pdfb_alphas *a, long long n, const double *q2, double *out,
                       cudaStream_t st, int q_is_q = 0);
int pdfb_setup_records(const double *d_z, IntervalRec *d_rec, IntervalRec32 *d_rec32, int n_arrays,
                       const int *h_off, cudaStream_t st);
int pdfb_setup_group_slices(const double *d_src, double *d_valg, int s_knot_off, int nx, int nx4, int nq,
                            int n_pid, int n_groups, long long group_stride, cudaStream_t st, int W, int n_members,
                            long long src_mstride);
int pdfb_smem_eligible(const pdfb_grid *g);
int pdfb_lumi_plan(pdfb_grid *g);
int pdfb_launch_xfxq2_smem(const pdfb_grid *g, int n_req, const int *cols, long long n, const double *x,
                           const double *q2, double *out, long long out_stride, cudaStream_t st, int mode,
                           int member0, int n_mem);
int pdfb_setup_ln(const double *d_raw, double *d_z, int n, cudaStream_t st);
int pdfb_setup_alphas_fast(const IntervalRec *d_rec, const double *d_a, const double *d_q2k, unsigned char *d_lines,
                           const double2 *d_lntab, int n_sub, const int *h_off, cudaStream_t st);
#define PDFB_ALPHAS_LINE 384   // bytes per interval in the fast-path image
int pdfb_setup_values(const double *d_src, double *d_dst, int nx, int nq, int n_pid, int kpad,
                      cudaStream_t st, int n_members, long long src_mstride, long long dst_mstride);

#define PDFB_CUDA(call)                          \
    do {                                         \
        cudaError_t e_ = (call);                 \
        if (e_ != cudaSuccess) return PDFB_ECUDA; \
    } while (0)
