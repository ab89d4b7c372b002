// lumi_kernels.cu -- pdf_lumi_events: the fused parton-luminosity call for Monte-Carlo integrands
// (section 4.1, 141-169 section 4.2: an event carries the two
// momentum fractions x1, x2 and ONE scale Q^2; ~1e6 events at once).
//
//   lumi[e] = sum_t coeff[t] * xf_{a_t}(x1_e, Q2_e) * xf_{b_t}(x2_e, Q2_e)        (optionally / (x1_e x2_e))
//
// where xf is exactly what pdf_xfxq2 returns (readings O3-O5).  The product couples flavours of
// different groups, so the flavour-group slices of the main kernel are of no use here: a CTA must
// hold ALL flavours of the rows it works on.  The table is therefore cut along Q^2 instead:
//   * a BAND of R consecutive Q^2 rows of every 2-column slice (R rows x nx2 knots x 16 B x NPAIR pairs,
//     ~200 KB) is staged by TMA bulk copies; it serves the cells c0 <= gi < c0 + R - 3;
//   * every CTA sweeps ITS OWN events once per band and evaluates those whose Q^2 falls into the band
//     (all CTAs do all bands: the load is balanced whatever the Q^2 distribution; events at q_min, a
//     quarter of config 5, do not pile up on one CTA);
//   * the events of a band are compacted per warp (ballot, shared-memory lists of coordinates) and
//     evaluated 32 at a time on full lanes: ln Q^2, the Q^2 interval and its four weights ONCE per
//     event, then per beam one x search and NPAIR 2-column stencil gathers (the conflict-free
//     row-pair pattern of xfxq2_smem.cuh) that share the sixteen products wu x wv;
//   * the bilinear form is contracted in registers (coefficients are constant-bank operands); 8 bytes
//     per event leave the SM instead of 176.
// Events with a point outside the grid (or all events of a grid the shared-memory path does not take)
// go through k_lumi_general: one thread per event, the read-only-cache evaluation of xfxq2_v0.cuh.
#include <cmath>
#include <cstring>

#include "xfxq2_smem.cuh"
#include "xfxq2_v0.cuh"

#define LUMI_NT 512
#define LUMI_LIST 64  // entries per warp list

// c[a][b]; need1 / need2: bit p set if beam 1 / beam 2 needs a column of pair p (a pair no term refers to is not gathered)
struct LumiCoef { double c[PDFB_LUMI_MAXF][PDFB_LUMI_MAXF]; unsigned need1, need2; };

// the sixteen products (x weight of the knot read at step s) x (v weight of its row), for one beam
struct Beam { uint32_t a[8]; double w[2][8]; };

__device__ __forceinline__ void make_beam(Beam &b, uint32_t row0, uint32_t RB, int node0, const double wu[4], const double vw[4], int lane8)
{
    const uint32_t base = row0 + (uint32_t)(node0 * 16);
    const int rho = (lane8 - (int)(base >> 4)) & 7;  // see stencil2 (xfxq2_smem.cuh)
    double Wr[4];
    rot4(wu, rho & 3, Wr);
#pragma unroll
    for (int s = 0; s < 8; s++) {
        const int v = (s + rho) & 7;
        const bool low = v >> 2;
        b.a[s] = base + (uint32_t)((v & 3) << 4) + (low ? RB : 0u);
        b.w[0][s] = Wr[s & 3] * (low ? vw[1] : vw[0]);
        b.w[1][s] = Wr[s & 3] * (low ? vw[3] : vw[2]);
    }
}

// both columns of pair p at the beam's point: 16 conflict-free LDS.128
__device__ __forceinline__ void pair_value(const Beam &b, uint32_t off, uint32_t RB2x2, double &y0, double &y1)
{
    y0 = 0.0; y1 = 0.0;
#pragma unroll
    for (int pp = 0; pp < 2; pp++) {
        double2 c[8];
#pragma unroll
        for (int s = 0; s < 8; s++) c[s] = lds128(b.a[s] + off + (pp ? RB2x2 : 0u));
#pragma unroll
        for (int s = 0; s < 8; s++) { y0 = fma(b.w[pp][s], c[s].x, y0); y1 = fma(b.w[pp][s], c[s].y, y1); }
    }
}

template <int NPAIR>
__global__ void __launch_bounds__(LUMI_NT, 1)
k_lumi_band(const __grid_constant__ GridDev g, const __grid_constant__ LumiCoef C, const __grid_constant__ LumiLayout L,
            long long n, const double *__restrict__ x1, const double *__restrict__ x2, const double *__restrict__ q2,
            double *__restrict__ out, int flags)
{
    constexpr int NF = 2 * NPAIR;
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) unsigned long long mbar;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, lane8 = tid & 7;
    const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(&mbar);
    const uint32_t band0 = s0 + (uint32_t)L.l_band, RB = (uint32_t)L.RB2;
    SmemViews sv;
    sv.tab = band0; sv.row_bytes = RB;
    sv.xrec = s0 + (uint32_t)g.a_xrec; sv.qrec = s0 + (uint32_t)L.l_qrec;
    sv.xk = reinterpret_cast<const double *>(smem + g.a_xk);
    sv.q2k = reinterpret_cast<const double *>(smem + g.a_q2k);
    sv.lutx = reinterpret_cast<const unsigned short *>(smem + g.a_lutx);
    sv.lutq = reinterpret_cast<const unsigned short *>(smem + g.a_lutq);
    // per-warp lists of the events waiting for a full batch
    double *lx1 = reinterpret_cast<double *>(smem + L.l_list) + warp * LUMI_LIST;
    double *lx2 = reinterpret_cast<double *>(smem + L.l_list) + (LUMI_NT / 32 + warp) * LUMI_LIST;
    double *lq = reinterpret_cast<double *>(smem + L.l_list) + (2 * (LUMI_NT / 32) + warp) * LUMI_LIST;
    uint32_t *le = reinterpret_cast<uint32_t *>(smem + L.l_list + 3 * (LUMI_NT / 32) * LUMI_LIST * 8) + warp * LUMI_LIST;

    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    {   // search tables and interval records (as in xfxq2_smem.cu); the whole band area starts out finite
        const int4 *src = reinterpret_cast<const int4 *>(g.aux);
        int4 *pre = reinterpret_cast<int4 *>(smem), *qr = reinterpret_cast<int4 *>(smem + L.l_qrec);
        const int npre = g.pre_bytes / 16, nqr = 128 * g.nq_tot / 16;
        for (int e = tid; e < npre; e += LUMI_NT) pre[e] = __ldg(src + e);
        for (int e = tid; e < nqr; e += LUMI_NT) qr[e] = __ldg(src + npre + e);
        int4 *bz = reinterpret_cast<int4 *>(smem + L.l_band);
        for (int e = tid; e < (L.l_qrec - L.l_band) / 16; e += LUMI_NT) bz[e] = make_int4(0, 0, 0, 0);  // the pairs' areas and the tail pad
#ifdef PDFB_CHECKED
        // poison what a band will overwrite (the rows of the pairs that exist): only a pair that does not exist
        // and the alignment row keep their zeros
        for (int p = 0; p < g.n_groups2; p++)
            for (int e = tid; e < L.R * L.RB2 / 8; e += LUMI_NT)
                reinterpret_cast<unsigned long long *>(smem + L.l_band + p * L.pair_stride)[e] = 0x7ff8dead00000000ULL;
#endif
    }
    const long long n_tiles = (n + LUMI_NT - 1) / LUMI_NT;
    for (int band = 0; band < L.n_bands; band++) {
        const int c0 = band * L.CB, c1 = min(c0 + L.CB, L.ncell);
        const int r0 = min(max(c0 - 1, 0), g.nq_tot - L.R);
        // generic-proxy writes (the zero fill, the previous band's reads) are ordered before the async copies
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (tid == 0) {
            const int bytes = L.R * L.RB2;
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(bytes * g.n_groups2) : "memory");
            for (int p = 0; p < g.n_groups2; p++) {
                const unsigned char *src = reinterpret_cast<const unsigned char *>(g.valg2) + (size_t)p * g.slice2_bytes + (size_t)r0 * L.RB2;
                for (int o = 0; o < bytes; o += 32768) {
                    const int nb = min(32768, bytes - o);
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(band0 + (uint32_t)(p * L.pair_stride + o)), "l"(src + o), "r"(nb), "r"(mb) : "memory");
                }
            }
        }
        {
            uint32_t done = 0;
            const uint32_t parity = band & 1;
            while (!done)
                asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                             : "=r"(done) : "r"(mb), "r"(parity) : "memory");
        }
        const double qlo = sv.q2k[c0], qhi = sv.q2k[c1];
        const bool last = (c1 == L.ncell);
        int cnt = 0;  // entries in this warp's list (warp-uniform)

        auto eval_batch = [&](int m) {  // the first m (<= 32) entries of the list, one per lane
            const bool act = lane < m;
            const double xa = act ? lx1[lane] : g.x_min, xb = act ? lx2[lane] : g.x_min, qv = act ? lq[lane] : qlo;
            const double v = ln_pos(qv);
            const int gi = locate_q(g, sv, qv, v);
            const IntervalRec32 rq = load_rec4(sv.qrec + (uint32_t)gi * 128u, lane8);
            double vw[4];
            weights_rec32(rq, (v - rq.z0) * rq.inv_dz, vw);
            const uint32_t row0 = band0 + (uint32_t)((gi - 1 - r0) * (int)RB);
            double h[NF];
            {   // beam 1, then h[b] = sum_a c[a][b] f_a(x1)
                const double u = ln_pos(xa);
                const int i = locate_x(g, sv, xa, u);
                const IntervalRec32 rx = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
                double wu[4];
                weights_rec32(rx, (u - rx.z0) * rx.inv_dz, wu);
                Beam bm;
                make_beam(bm, row0, RB, i - 1, wu, vw, lane8);
#pragma unroll
                for (int b = 0; b < NF; b++) h[b] = 0.0;
#pragma unroll
                for (int p = 0; p < NPAIR; p++) {
                    if (!((C.need1 >> p) & 1)) continue;  // uniform: no term takes a flavour of this pair from beam 1
                    double f0, f1;
                    pair_value(bm, (uint32_t)(p * L.pair_stride), 2u * RB, f0, f1);
#pragma unroll
                    for (int b = 0; b < NF; b++) h[b] = fma(C.c[2 * p + 1][b], f1, fma(C.c[2 * p][b], f0, h[b]));
                }
            }
            double lum = 0.0;
            {   // beam 2
                const double u = ln_pos(xb);
                const int i = locate_x(g, sv, xb, u);
                const IntervalRec32 rx = load_rec4(sv.xrec + (uint32_t)i * 128u, lane8);
                double wu[4];
                weights_rec32(rx, (u - rx.z0) * rx.inv_dz, wu);
                Beam bm;
                make_beam(bm, row0, RB, i - 1, wu, vw, lane8);
#pragma unroll
                for (int p = 0; p < NPAIR; p++) {
                    if (!((C.need2 >> p) & 1)) continue;
                    double f0, f1;
                    pair_value(bm, (uint32_t)(p * L.pair_stride), 2u * RB, f0, f1);
                    lum = fma(h[2 * p + 1], f1, fma(h[2 * p], f0, lum));
                }
            }
            if (flags & 1) lum /= xa * xb;
            if (act) __stcs(out + le[lane], lum);
        };

        double xa = 1.0, xb = 1.0, qv = 0.0;
        long long tile = blockIdx.x;
        if (tile < n_tiles) {
            const long long e = tile * LUMI_NT + tid;
            if (e < n) { xa = __ldg(x1 + e); xb = __ldg(x2 + e); qv = __ldg(q2 + e); }
        }
        for (; tile < n_tiles; tile += gridDim.x) {
            const long long e = tile * LUMI_NT + tid;
            double xan = 1.0, xbn = 1.0, qn = 0.0;  // next tile's coordinates in flight
            const long long en = e + (long long)gridDim.x * LUMI_NT;
            if (en < n) { xan = __ldg(x1 + en); xbn = __ldg(x2 + en); qn = __ldg(q2 + en); }
            const bool in_grid = e < n && xa >= g.x_min && xa <= g.x_max && xb >= g.x_min && xb <= g.x_max &&
                                 qv >= g.q2_min && qv <= g.q2_max;
            const bool mine = in_grid && qv >= qlo && (last ? true : qv < qhi);
            const unsigned m = __ballot_sync(0xffffffffu, mine);
            if (m) {
                if (mine) {
                    const int pos = cnt + __popc(m & ((1u << lane) - 1u));
                    PDFB_ASSERT(pos < LUMI_LIST);
                    lx1[pos] = xa; lx2[pos] = xb; lq[pos] = qv; le[pos] = (uint32_t)e;
                }
                cnt += __popc(m);
                __syncwarp();
                if (cnt >= 32) {
                    eval_batch(32);
                    __syncwarp();
                    const int rem = cnt - 32;  // < 32: moved to the front
                    double t1 = 0.0, t2 = 0.0, t3 = 0.0;
                    uint32_t t4 = 0;
                    if (lane < rem) { t1 = lx1[32 + lane]; t2 = lx2[32 + lane]; t3 = lq[32 + lane]; t4 = le[32 + lane]; }
                    __syncwarp();
                    if (lane < rem) { lx1[lane] = t1; lx2[lane] = t2; lq[lane] = t3; le[lane] = t4; }
                    __syncwarp();
                    cnt = rem;
                }
            }
            xa = xan; xb = xbn; qv = qn;
        }
        if (cnt) { eval_batch(cnt); __syncwarp(); }
    }
}

// Events the band kernel does not take: a point outside the grid, a coordinate without a value, or a
// grid without the shared-memory path (all == 1: every event).  One thread per event.
__global__ void __launch_bounds__(128, 8)  // few registers: the usual case is a scan that finds nothing to do
k_lumi_general(const __grid_constant__ GridDev g, const __grid_constant__ LumiCoef C, int nf, int all, long long n, const double *__restrict__ x1,
               const double *__restrict__ x2, const double *__restrict__ q2, double *__restrict__ out, int flags)
{
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n) return;
    const double xa = x1[e], xb = x2[e], qv = q2[e];
    const bool in_grid = xa >= g.x_min && xa <= g.x_max && xb >= g.x_min && xb <= g.x_max && qv >= g.q2_min && qv <= g.q2_max;
    if (in_grid && !all) return;
    ReqCols rc;
    rc.n = nf;
    for (int k = 0; k < nf; k++) rc.col[k] = k;
    // beam 2 first: hv[a] = sum_b c[a][b] xf_b(x2); then beam 1 into the same array and the sum over a
    double f[PDFB_LUMI_MAXF], hv[PDFB_LUMI_MAXF];
    const bool ok2 = xf_point_v0(g, g.val, rc, xb, qv, f);
    for (int a = 0; a < nf; a++) {
        double h = 0.0;
        for (int b = 0; b < nf; b++) h = fma(C.c[a][b], f[b], h);
        hv[a] = h;
    }
    const bool ok1 = xf_point_v0(g, g.val, rc, xa, qv, f);
    double lum = 0.0;
    for (int a = 0; a < nf; a++) lum = fma(f[a], hv[a], lum);
    if (flags & 1) lum /= xa * xb;
    if (!ok1 || !ok2) {
        lum = __longlong_as_double(0x7ff8000000000000LL);
        atomicAdd(g.n_invalid, 1ULL);
    }
    out[e] = lum;
}

// ------------------------------------------------------------------------------ host side
static const int LUMI_STATIC_SMEM = 256;

// Band plan of a handle (at load): how many Q^2 rows of all 2-column slices fit shared memory.
int pdfb_lumi_plan(pdfb_grid *g)
{
    LumiLayout &L = g->lumi;
    memset(&L, 0, sizeof(L));
    g->lumi_npair = 0;
    const GridDev &d = g->d;
    if (!(d.smem_ok & 2)) return PDFB_OK;  // no 2-column slices: general kernel only (a set: its member 0)
    int npair = 0;
    for (int c : {2, 4, 6, 7}) if (d.n_groups2 <= c) { npair = c; break; }
    if (!npair) return PDFB_OK;
    int dev_max = 0;
    if (cudaDeviceGetAttribute(&dev_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, g->device) != cudaSuccess) return PDFB_OK;
    L.RB2 = d.nx2 * 16;
    L.ncell = d.nq_tot - 1;
    const int qrec_bytes = 128 * d.nq_tot;
    const int list_bytes = (LUMI_NT / 32) * LUMI_LIST * (3 * 8 + 4);
    // the stencil of the last knot's phantom interval (xfxq2_smem.cuh) reaches two rows and three knots past a pair's
    // rows with weight 0: the next pair's rows for all pairs but the last, a pad of zeros after the last
    const int tail_pad = (2 * L.RB2 + 3 * 16 + 127) & ~127;
    const int avail = dev_max - LUMI_STATIC_SMEM - d.pre_bytes - qrec_bytes - list_bytes - tail_pad - 256;
    int R = avail / (npair * L.RB2);
    R &= ~1;                                   // even: the pair stride stays a multiple of 128 bytes
    if (R >= d.nq_tot) { L.R = d.nq_tot; L.R_alloc = (d.nq_tot + 1) & ~1; L.CB = L.ncell; }
    else { L.R = L.R_alloc = R; L.CB = R - 3; }
    if (L.R < 4 || L.CB < 1) return PDFB_OK;
    L.n_bands = (L.ncell + L.CB - 1) / L.CB;
    L.pair_stride = L.R_alloc * L.RB2;
    L.l_band = d.pre_bytes;                    // 128-byte aligned (pre ends with the 128-byte xrec lines)
    L.l_qrec = L.l_band + npair * L.pair_stride + tail_pad;
    L.l_list = L.l_qrec + qrec_bytes;
    L.total = L.l_list + list_bytes;
    if (L.total + LUMI_STATIC_SMEM > dev_max || (L.pair_stride & 127) || (L.l_band & 127)) return PDFB_OK;
    cudaError_t e = cudaSuccess;
    const int lim = dev_max - LUMI_STATIC_SMEM;
    if (npair == 2) e = cudaFuncSetAttribute(k_lumi_band<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
    if (npair == 4) e = cudaFuncSetAttribute(k_lumi_band<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
    if (npair == 6) e = cudaFuncSetAttribute(k_lumi_band<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
    if (npair == 7) e = cudaFuncSetAttribute(k_lumi_band<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim);
    if (e != cudaSuccess) { cudaGetLastError(); return PDFB_OK; }
    g->lumi_npair = npair;
    return PDFB_OK;
}

extern "C" int pdf_lumi_events(const pdfb_grid *g, const pdfb_alphas *a, int n_terms, const int *pid_a, const int *pid_b,
                               const double *coeff, long long n, const double *x1, const double *x2, const double *q2,
                               double *lumi, double *alphas_out, int flags, void *cuda_stream)
{
    if (!g || n < 0 || n_terms < 1 || !pid_a || !pid_b || !coeff) return PDFB_EINVAL;
    if (n > 0 && (!x1 || !x2 || !q2 || !lumi)) return PDFB_EINVAL;
    if ((a == nullptr) != (alphas_out == nullptr)) return PDFB_EINVAL;
    if (a && a->device != g->device) return PDFB_EINVAL;
    if (g->d.n_pid > PDFB_LUMI_MAXF) return PDFB_ELIMIT;
    LumiCoef C;
    memset(&C, 0, sizeof(C));
    for (int t = 0; t < n_terms; t++) {
        int ca = -1, cb = -1;
        const int pa = pid_a[t] == 0 ? 21 : pid_a[t], pb = pid_b[t] == 0 ? 21 : pid_b[t];
        for (int k = 0; k < g->d.n_pid; k++) { if (g->pids[k] == pa) ca = k; if (g->pids[k] == pb) cb = k; }
        if (ca < 0 || cb < 0) return PDFB_EPID;
        if (!std::isfinite(coeff[t])) return PDFB_EINVAL;
        C.c[ca][cb] += coeff[t];
        C.need1 |= 1u << (ca >> 1); C.need2 |= 1u << (cb >> 1);
    }
    if (n == 0) return PDFB_OK;
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long long SLICE = 1LL << 31;  // event indices travel as 32-bit offsets
    for (long long off = 0; off < n; off += SLICE) {
        const long long m = (n - off < SLICE) ? (n - off) : SLICE;
        const int band = g->lumi_npair;
        if (band) {
            long long tiles = (m + LUMI_NT - 1) / LUMI_NT;
            const unsigned grid = (unsigned)(tiles < g->sms ? tiles : g->sms);
#define LUMI_LAUNCH(NP) k_lumi_band<NP><<<grid, LUMI_NT, g->lumi.total, st>>>(g->d, C, g->lumi, m, x1 + off, x2 + off, q2 + off, lumi + off, flags)
            if (band == 2) LUMI_LAUNCH(2); else if (band == 4) LUMI_LAUNCH(4); else if (band == 6) LUMI_LAUNCH(6); else LUMI_LAUNCH(7);
#undef LUMI_LAUNCH
            pdfb_count_launch(1);
        }
        k_lumi_general<<<(unsigned)((m + 127) / 128), 128, 0, st>>>(g->d, C, g->d.n_pid, band ? 0 : 1, m, x1 + off, x2 + off, q2 + off, lumi + off, flags);
        pdfb_count_launch(1);
    }
    PDFB_CUDA(cudaGetLastError());
    if (a) return pdfb_launch_alphas(a, n, q2, alphas_out, st);
    return PDFB_OK;
}
