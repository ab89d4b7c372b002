// xfxq2_smem.cu -- K2/K3, the shared-memory path of pdf_xfxq2 (readings O3-O5).
//
// Why it looks the way it does ("Kernel design"): per point and flavour the method
// gathers a 4x4 value stencil -- 1408 B of table per point at 11 flavours against 104 B of HBM
// traffic -- and the points of a warp almost never share a cell.  The gather is what bounds the
// kernel, so it is fed from shared memory at full crossbar width, with no bank conflict:
//   * the value table is split into FLAVOUR GROUPS of 4 columns; one group's slice
//     [s][iq][ix4][4] (32 B per knot) fits shared memory and is staged once per CTA by TMA bulk
//     copies.  Each persistent CTA serves one group for all points of its tiles, so it writes
//     whole flavour rows with coalesced stores and no point ever has to be re-ordered;
//   * one stencil row (4 knots x 4 flavours) is 128 contiguous bytes = 8 chunks of 16 B that
//     cover all 8 bank groups.  Lane l reads them in the rotated order c = (s + l - 2*node0) & 7,
//     so at every step the 8 lanes of a quarter-warp hit 8 distinct bank groups whatever cells
//     their points fell in: 32 conflict-free LDS.128 per point and group, 4 wavefronts;
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

#define NT_SMEM 512

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ double cont_e(double r, double yL, double yH)  // reading O4
{
    if (yL > 1e-3 && yH > 1e-3) {
        double lL = log(yL);
        return exp(fma(r, log(yH) - lL, lL));
    }
    return fma(r, yH - yL, yL);
}

// window of 4 knots containing m-1..m+2 shifted into [0, M-1] (M >= 4); weights follow
__device__ __forceinline__ int shift_set(int m, int M, double w[4])
{
    int base = m - 1;
    if (base < 0) {            // m == 0: knot -1 carries weight exactly 0
        w[0] = w[1]; w[1] = w[2]; w[2] = w[3]; w[3] = 0.0;
        base = 0;
    } else if (base + 3 > M - 1) {  // m == M-2: knot M carries weight exactly 0
        w[3] = w[2]; w[2] = w[1]; w[1] = w[0]; w[0] = 0.0;
        base = M - 4;
    }
    return base;
}

__device__ __forceinline__ void weights_rec32(const IntervalRec32 &r, double t, double w[4])
{
    double t2 = t * t, t3 = t2 * t;
    double h01 = 3.0 * t2 - 2.0 * t3;
    double h00 = 1.0 - h01;
    double h11 = t3 - t2;
    double h10 = h11 - t2 + t;
    double aL1 = (r.aLm == 0.0) ? 1.0 : 0.5, aH0 = (r.aHp == 0.0) ? -1.0 : -0.5;
    double aL0 = -(r.aLm + aL1), aH1 = -(aH0 + r.aHp);
    w[0] = h10 * r.aLm;
    w[1] = fma(h11, aH0, fma(h10, aL0, h00));
    w[2] = fma(h11, aH1, fma(h10, aL1, h01));
    w[3] = h11 * r.aHp;
}

// x-direction state of one point: smem byte offset of knot node0 within a table row, the
// rotated chunk offsets and the x weights in rotated order
struct USet { uint32_t off[8]; double wrot[8]; int rot; };

__device__ __forceinline__ void make_uset(USet &u, int node0, const double w[4], int lane8)
{
    int rot = (lane8 - 2 * node0) & 7;
    u.rot = rot;
#pragma unroll
    for (int s = 0; s < 8; s++) u.off[s] = (uint32_t)(node0 * 32 + (((s + rot) & 7) << 4));
    // wrot[s] = w[((s + rot) & 7) >> 1]: barrel rotation of {w0,w0,w1,w1,w2,w2,w3,w3}
    double a[8] = {w[0], w[0], w[1], w[1], w[2], w[2], w[3], w[3]}, b[8];
#pragma unroll
    for (int s = 0; s < 8; s++) b[s] = (rot & 1) ? a[(s + 1) & 7] : a[s];
#pragma unroll
    for (int s = 0; s < 8; s++) a[s] = (rot & 2) ? b[(s + 2) & 7] : b[s];
#pragma unroll
    for (int s = 0; s < 8; s++) u.wrot[s] = (rot & 4) ? a[(s + 4) & 7] : a[s];
}

// sum_b wv[b] * sum_a wu[a] * V[row0+b][node0+a][0..3] -> y[4]
__device__ __forceinline__ void gather4(uint32_t tab, uint32_t row_bytes, int row0, const USet &u,
                                        const double wv[4], double y[4])
{
    double2 tE = make_double2(0.0, 0.0), tO = make_double2(0.0, 0.0);
    uint32_t base = tab + (uint32_t)row0 * row_bytes;
#pragma unroll
    for (int b = 0; b < 4; b++) {
        double2 E = make_double2(0.0, 0.0), O = make_double2(0.0, 0.0);
#pragma unroll
        for (int s = 0; s < 8; s += 2) {
            double2 v0 = lds128(base + u.off[s]), v1 = lds128(base + u.off[s + 1]);
            E.x = fma(u.wrot[s], v0.x, E.x); E.y = fma(u.wrot[s], v0.y, E.y);
            O.x = fma(u.wrot[s + 1], v1.x, O.x); O.y = fma(u.wrot[s + 1], v1.y, O.y);
        }
        tE.x = fma(wv[b], E.x, tE.x); tE.y = fma(wv[b], E.y, tE.y);
        tO.x = fma(wv[b], O.x, tO.x); tO.y = fma(wv[b], O.y, tO.y);
        base += row_bytes;
    }
    // even steps carried chunk parity (rot & 1): chunk parity 0 = columns 0,1; 1 = columns 2,3
    bool sw = u.rot & 1;
    y[0] = sw ? tO.x : tE.x; y[1] = sw ? tO.y : tE.y;
    y[2] = sw ? tE.x : tO.x; y[3] = sw ? tE.y : tO.y;
}

struct SmemViews {
    uint32_t tab, row_bytes;
    const double *xk, *q2k;
    const IntervalRec32 *xrec, *qrec;
    const unsigned short *lutx, *lutq;
    const unsigned char *subof;
};

// points outside the grid (readings O4/O5): up to 2 x-sets times 2 v-sets
__device__ __noinline__ void slow_point(const GridDev &g, const SmemViews &sv, double xv, double qv,
                                        int lane8, double res[4])
{
    const bool low_x = xv < g.x_min, high_q = qv > g.q2_max, low_q = qv < g.q2_min;
    USet u1, u2;
    double rA = 0.0;
    if (!low_x) {
        double u = log(xv);
        int b = min(max((int)((u - g.lutx_u0) * g.lutx_inv_h), 0), PDFB_LUT_BINS - 1);
        int i = sv.lutx[b];
        while (i < g.nx - 2 && sv.xk[i + 1] <= xv) ++i;
        while (i > 0 && sv.xk[i] > xv) --i;
        IntervalRec32 r = sv.xrec[i];
        double w[4];
        weights_rec32(r, (u - r.z0) * r.inv_dz, w);
        int node0 = shift_set(i, g.nx, w);
        make_uset(u1, node0, w, lane8);
    } else {  // rule A: one-hot sets on knots 0 and 1
        rA = (log(xv) - g.U0) * g.inv_dU01;
        double e0[4] = {1.0, 0.0, 0.0, 0.0}, e1[4] = {0.0, 1.0, 0.0, 0.0};
        make_uset(u1, 0, e0, lane8);
        make_uset(u2, 0, e1, lane8);
    }
    double wv1[4], wv2[4] = {0.0, 0.0, 0.0, 0.0};
    int row1, row2 = 0;
    double rB = 0.0;
    if (high_q) {  // the last two Q^2 knots of the last sub-grid
        rB = (log(qv) - g.Va) * g.inv_dVab;
        row1 = row2 = g.nq_tot - 4;
        wv1[0] = wv1[1] = wv1[3] = 0.0; wv1[2] = 1.0;
        wv2[0] = wv2[1] = wv2[2] = 0.0; wv2[3] = 1.0;
    } else if (low_q) {  // q_min (knot 0 of sub-grid 0) and 1.01 q_min
        row1 = 0;
        wv1[0] = 1.0; wv1[1] = wv1[2] = wv1[3] = 0.0;
#pragma unroll
        for (int b = 0; b < 4; b++) wv2[b] = g.wvC[b];
        row2 = shift_set(g.jC, g.q_off[1], wv2);
    } else {
        double v = log(qv);
        int b = min(max((int)((v - g.lutq_v0) * g.lutq_inv_h), 0), PDFB_LUT_BINS - 1);
        int m = sv.lutq[b];
        while (m < g.nq_tot - 1 && sv.q2k[m + 1] <= qv) ++m;
        while (m > 0 && sv.q2k[m] > qv) --m;
        int s = sv.subof[m];
        int nq = g.q_off[s + 1] - g.q_off[s];
        int j = min(m - g.q_off[s], nq - 2);
        IntervalRec32 r = sv.qrec[g.q_off[s] + j];
        weights_rec32(r, (v - r.z0) * r.inv_dz, wv1);
        row1 = g.q_off[s] + shift_set(j, nq, wv1);
    }
    const bool two_v = high_q || low_q;
    double y1[4], y2[4] = {0.0, 0.0, 0.0, 0.0};
    gather4(sv.tab, sv.row_bytes, row1, u1, wv1, y1);
    if (two_v) gather4(sv.tab, sv.row_bytes, row2, u1, wv2, y2);
    if (low_x) {
        double h1[4], h2[4];
        gather4(sv.tab, sv.row_bytes, row1, u2, wv1, h1);
#pragma unroll
        for (int k = 0; k < 4; k++) y1[k] = cont_e(rA, y1[k], h1[k]);
        if (two_v) {
            gather4(sv.tab, sv.row_bytes, row2, u2, wv2, h2);
#pragma unroll
            for (int k = 0; k < 4; k++) y2[k] = cont_e(rA, y2[k], h2[k]);
        }
    }
    const double rho = qv / g.q2_min;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        double r = y1[k];
        if (high_q) {
            r = cont_e(rB, y1[k], y2[k]);
        } else if (low_q) {
            double gamma = 0.0;
            if (fabs(y1[k]) >= 1e-5) gamma = fmax(-2.5, (y2[k] - y1[k]) / y1[k] / 0.01);
            r = y1[k] * pow(rho, fma(gamma, rho, 1.0 - rho));
        }
        res[k] = r;
    }
}

__global__ void __launch_bounds__(NT_SMEM, 1)
k_xfxq2_smem(const GridDev g, const PassList pl, long long n, const double *__restrict__ x,
             const double *__restrict__ q2, double *__restrict__ out, long long out_stride)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) unsigned long long mbar;
    const int tid = threadIdx.x;
    const int pass = blockIdx.x % pl.n, seq = blockIdx.x / pl.n, nseq = gridDim.x / pl.n;
    if (seq >= nseq) return;
    unsigned char *s_aux = smem + g.slice_bytes;
    const uint32_t tab = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t mb = (uint32_t)__cvta_generic_to_shared(&mbar);

    // ---- stage this CTA's flavour-group slice with TMA bulk copies; small tables by plain loads
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mb));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mb), "r"(g.slice_bytes) : "memory");
        const unsigned char *src = reinterpret_cast<const unsigned char *>(g.valg) + (size_t)pl.group[pass] * g.slice_bytes;
        for (int o = 0; o < g.slice_bytes; o += 32768) {
            int bytes = min(32768, g.slice_bytes - o);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(tab + o), "l"(src + o), "r"(bytes), "r"(mb) : "memory");
        }
    }
    for (int e = tid; e < g.aux_bytes / 16; e += NT_SMEM)
        reinterpret_cast<int4 *>(s_aux)[e] = __ldg(reinterpret_cast<const int4 *>(g.aux) + e);
    __syncthreads();
    {
        uint32_t done = 0;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }"
                         : "=r"(done) : "r"(mb) : "memory");
    }
    SmemViews sv;
    sv.tab = tab; sv.row_bytes = (uint32_t)g.nx4 * 32u;
    sv.xk = reinterpret_cast<const double *>(s_aux + g.a_xk);
    sv.q2k = reinterpret_cast<const double *>(s_aux + g.a_q2k);
    sv.xrec = reinterpret_cast<const IntervalRec32 *>(s_aux + g.a_xrec);
    sv.qrec = reinterpret_cast<const IntervalRec32 *>(s_aux + g.a_qrec);
    sv.lutx = reinterpret_cast<const unsigned short *>(s_aux + g.a_lutx);
    sv.lutq = reinterpret_cast<const unsigned short *>(s_aux + g.a_lutq);
    sv.subof = s_aux + g.a_subof;
    const int lane8 = tid & 7;
    const int r0 = pl.row[pass][0], r1 = pl.row[pass][1], r2 = pl.row[pass][2], r3 = pl.row[pass][3];

    for (long long tile = seq; tile * NT_SMEM < n; tile += nseq) {
        const long long p = tile * NT_SMEM + tid;
        if (p >= n) continue;
        const double xv = __ldg(x + p), qv = __ldg(q2 + p);
        double y[4];
        if (xv >= g.x_min && xv <= g.x_max && qv >= g.q2_min && qv <= g.q2_max) {
            // ---- in range: locate (LUT guess + exact comparisons), weights, one gather
            const double u = log(xv), v = log(qv);
            int b = min(max((int)((u - g.lutx_u0) * g.lutx_inv_h), 0), PDFB_LUT_BINS - 1);
            int i = sv.lutx[b];
            while (i < g.nx - 2 && sv.xk[i + 1] <= xv) ++i;
            while (i > 0 && sv.xk[i] > xv) --i;
            b = min(max((int)((v - g.lutq_v0) * g.lutq_inv_h), 0), PDFB_LUT_BINS - 1);
            int m = sv.lutq[b];
            while (m < g.nq_tot - 1 && sv.q2k[m + 1] <= qv) ++m;
            while (m > 0 && sv.q2k[m] > qv) --m;
            const int s = sv.subof[m];
            const int qo = g.q_off[s], nq = g.q_off[s + 1] - qo;
            const int j = min(m - qo, nq - 2);
            const IntervalRec32 rx = sv.xrec[i], rq = sv.qrec[qo + j];
            double wu[4], wv[4];
            weights_rec32(rx, (u - rx.z0) * rx.inv_dz, wu);
            weights_rec32(rq, (v - rq.z0) * rq.inv_dz, wv);
            const int node0 = shift_set(i, g.nx, wu);
            const int row0 = qo + shift_set(j, nq, wv);
            USet us;
            make_uset(us, node0, wu, lane8);
            gather4(tab, sv.row_bytes, row0, us, wv, y);
        } else if (!(xv > 0.0) || !(qv > 0.0) || !(xv <= g.x_max) || isinf(qv)) {
            y[0] = y[1] = y[2] = y[3] = __longlong_as_double(0x7ff8000000000000LL);
            if (pass == 0) atomicAdd(g.n_invalid, 1ULL);
        } else {
            slow_point(g, sv, xv, qv, lane8, y);
        }
        if (r0 >= 0) __stcs(out + r0 * out_stride + p, y[0]);
        if (r1 >= 0) __stcs(out + r1 * out_stride + p, y[1]);
        if (r2 >= 0) __stcs(out + r2 * out_stride + p, y[2]);
        if (r3 >= 0) __stcs(out + r3 * out_stride + p, y[3]);
    }
}

static int smem_needed(const GridDev &d) { return d.slice_bytes + d.aux_bytes; }

int pdfb_smem_eligible(const pdfb_grid *g)
{
    if (getenv("PDFB_FORCE_FALLBACK")) return 0;  // testing: force the read-only-cache path
    int dev_max = 0;
    if (cudaDeviceGetAttribute(&dev_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, g->device) != cudaSuccess) return 0;
    if (smem_needed(g->d) + 1024 > dev_max) return 0;
    // the attribute is per function, not per handle: raise it once to the device maximum
    static int attr_set_for = -1;
    if (attr_set_for != g->device) {
        if (cudaFuncSetAttribute(k_xfxq2_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, dev_max - 1024) != cudaSuccess) {
            cudaGetLastError();
            return 0;
        }
        attr_set_for = g->device;
    }
    return 1;
}

int pdfb_launch_xfxq2_smem(const pdfb_grid *g, int n_req, const int *cols, long long n, const double *x,
                           const double *q2, double *out, long long out_stride, cudaStream_t st)
{
    // passes: one per (flavour group, distinct use of its columns); duplicates get extra passes
    PassList pl;
    pl.n = 0;
    bool used[PDFB_MAX_PIDS] = {false};
    for (int left = n_req; left > 0;) {
        for (int grp = 0; grp < g->d.n_groups && left > 0; grp++) {
            int row[4] = {-1, -1, -1, -1}, hit = 0;
            for (int r = 0; r < n_req; r++)
                if (!used[r] && cols[r] / 4 == grp && row[cols[r] & 3] < 0) { row[cols[r] & 3] = r; used[r] = true; hit++; }
            if (!hit) continue;
            if (pl.n >= PDFB_MAX_PIDS) return PDFB_ELIMIT;
            pl.group[pl.n] = grp;
            for (int k = 0; k < 4; k++) pl.row[pl.n][k] = row[k];
            pl.n++;
            left -= hit;
        }
    }
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device);
    int per_pass = sms / pl.n;
    if (per_pass < 1) per_pass = 1;
    long long tiles = (n + NT_SMEM - 1) / NT_SMEM;
    if (per_pass > tiles) per_pass = (int)tiles;
    k_xfxq2_smem<<<per_pass * pl.n, NT_SMEM, smem_needed(g->d), st>>>(g->d, pl, n, x, q2, out, out_stride);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
