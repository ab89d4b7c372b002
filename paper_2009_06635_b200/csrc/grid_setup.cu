// grid_setup.cu -- K1: the grid-setup kernels, run once per pdf_grid_load / alphas_grid_load.
//
// Reading O2 ("special care ... close to quark mass thresholds and
// grids x edges, where the minimum number of knots required for bicubic interpolation is not
// available"): the derivative at a knot is the one-sided slope at either end of the knot
// array -- the x-knot array, or the Q^2 knots of ONE sub-grid -- and the plain mean of the two
// one-sided slopes inside.  K1 turns that rule into per-interval coefficient records
// (IntervalRec) so that a query only fetches Hermite coefficients, and re-lays the value
// table out for the evaluation kernel.
#include "pdfb_internal.cuh"

// natural logs of the knots, with the same function the queries use (reading R-ln)
__global__ void k1_ln_knots(const double *__restrict__ raw, double *__restrict__ z, int n)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) z[i] = pdfb_ln(raw[i]);
}

int pdfb_setup_ln(const double *d_raw, double *d_z, int n, cudaStream_t st)
{
    k1_ln_knots<<<(n + 127) / 128, 128, 0, st>>>(d_raw, d_z, n);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}

extern "C" int pdfb_debug_ln(const double *d_in, double *d_out, long long n, void *cuda_stream)
{
    if (!d_in || !d_out || n < 0 || n > 0x7fffffff) return PDFB_EINVAL;
    if (n == 0) return PDFB_OK;
    return pdfb_setup_ln(d_in, d_out, (int)n, (cudaStream_t)cuda_stream);
}

// One thread per interval m of the knot array z[0..M-1] (natural logs of the knots).
__global__ void k1_interval_records(const double *__restrict__ z, IntervalRec *__restrict__ rec,
                                    IntervalRec32 *__restrict__ rec32, int M)
{
    int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= M - 1) {
        if (m == M - 1) {  // pad entry so every knot index has a record; never used by a cell
            IntervalRec r = {z[m], 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
            rec[m] = r;
            if (rec32) { IntervalRec32 q = {z[m], 0.0, 0.0, 0.0}; for (int k = 0; k < 4; k++) rec32[4 * m + k] = q; }
        }
        return;
    }
    double dz = z[m + 1] - z[m];
    IntervalRec r;
    r.z0 = z[m];
    r.inv_dz = 1.0 / dz;
    if (m == 0) {  // one-sided: dz * d_m = y_{m+1} - y_m
        r.aLm = 0.0; r.aL0 = -1.0; r.aL1 = 1.0;
    } else {       // dz * d_m = 1/2 [ (y_{m+1}-y_m) + (dz/dz_left)(y_m - y_{m-1}) ]
        double rho = dz / (z[m] - z[m - 1]);
        r.aLm = -0.5 * rho; r.aL0 = 0.5 * (rho - 1.0); r.aL1 = 0.5;
    }
    if (m + 1 == M - 1) {
        r.aH0 = -1.0; r.aH1 = 1.0; r.aHp = 0.0;
    } else {       // dz * d_{m+1} = 1/2 [ (dz/dz_right)(y_{m+2}-y_{m+1}) + (y_{m+1}-y_m) ]
        double rho = dz / (z[m + 2] - z[m + 1]);
        r.aH0 = -0.5; r.aH1 = 0.5 * (1.0 - rho); r.aHp = 0.5 * rho;
    }
    rec[m] = r;
    if (rec32) {  // 4 copies = one 128-byte line: the 8 lanes of a quarter-warp read distinct bank groups
        IntervalRec32 q = {r.z0, r.inv_dz, r.aLm, r.aHp};
        for (int k = 0; k < 4; k++) rec32[4 * m + k] = q;
    }
}

// values of one sub-grid: file order [ix][iq][ipid] -> flavour-group slices [g][iq][nxp][W]
// (the shared-memory path stages one slice per CTA; W = 4 or 2 columns per group, nxp = padded
// knots per row); padding columns / knots = 0
__global__ void k1_group_slices(const double *__restrict__ src, double *__restrict__ valg, int s_knot_off,
                                int nx, int nxp, int nq, int n_pid, int n_groups, long long group_stride, int W,
                                long long src_mstride)
{
    src += blockIdx.y * src_mstride;                      // blockIdx.y = member of the set
    valg += blockIdx.y * (long long)n_groups * group_stride;
    long long tot = (long long)n_groups * nq * nxp * W;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < tot;
         e += (long long)gridDim.x * blockDim.x) {
        int slot = (int)(e % W);
        long long r = e / W;
        int ix = (int)(r % nxp); r /= nxp;
        int iq = (int)(r % nq);
        int grp = (int)(r / nq);
        int k = grp * W + slot;
        double v = (ix < nx && k < n_pid) ? src[((long long)ix * nq + iq) * n_pid + k] : 0.0;
        valg[grp * group_stride + ((long long)(s_knot_off + iq * nxp + ix)) * W + slot] = v;
    }
}

// values of one sub-grid: file order [ix][iq][ipid] -> [iq][ix][kpad], padding columns = 0
__global__ void k1_relayout_values(const double *__restrict__ src, double *__restrict__ dst, int nx,
                                   int nq, int n_pid, int kpad, long long src_mstride, long long dst_mstride)
{
    src += blockIdx.y * src_mstride;                      // blockIdx.y = member of the set
    dst += blockIdx.y * dst_mstride;
    long long tot = (long long)nx * nq * kpad;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < tot;
         e += (long long)gridDim.x * blockDim.x) {
        int k = (int)(e % kpad);
        long long knot = e / kpad;
        int ix = (int)(knot % nx), iq = (int)(knot / nx);
        dst[e] = (k < n_pid) ? src[((long long)ix * nq + iq) * n_pid + k] : 0.0;
    }
}

int pdfb_setup_records(const double *d_z, IntervalRec *d_rec, IntervalRec32 *d_rec32, int n_arrays,
                       const int *h_off, cudaStream_t st)
{
    for (int a = 0; a < n_arrays; a++) {
        int M = h_off[a + 1] - h_off[a];
        k1_interval_records<<<(M + 127) / 128, 128, 0, st>>>(d_z + h_off[a], d_rec + h_off[a],
                                                             d_rec32 ? d_rec32 + 4 * h_off[a] : nullptr, M);
        pdfb_count_launch(1);
    }
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}

int pdfb_setup_values(const double *d_src, double *d_dst, int nx, int nq, int n_pid, int kpad,
                      cudaStream_t st, int n_members, long long src_mstride, long long dst_mstride)
{
    long long tot = (long long)nx * nq * kpad;
    int blocks = (int)((tot + 255) / 256);
    if (blocks > 1184) blocks = 1184;
    k1_relayout_values<<<dim3(blocks, n_members), 256, 0, st>>>(d_src, d_dst, nx, nq, n_pid, kpad, src_mstride, dst_mstride);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}

int pdfb_setup_group_slices(const double *d_src, double *d_valg, int s_knot_off, int nx, int nx4, int nq,
                            int n_pid, int n_groups, long long group_stride, cudaStream_t st, int W, int n_members,
                            long long src_mstride)
{
    long long tot = (long long)n_groups * nq * nx4 * W;
    int blocks = (int)((tot + 255) / 256);
    if (blocks > 1184) blocks = 1184;
    k1_group_slices<<<dim3(blocks, n_members), 256, 0, st>>>(d_src, d_valg, s_knot_off, nx, nx4, nq, n_pid, n_groups, group_stride, W, src_mstride);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}

// alpha_s fast-path records: cubic coefficients of each interval in s = ln Q^2 - Z_m, from the O2 records.
// p(t) = h00 y0 + h10 dL + h01 y1 + h11 dH = y0 + dL t + (3(y1-y0) - 2 dL - dH) t^2 + (dL + dH - 2(y1-y0)) t^3,
// t = s / dZ: alpha_s(s) = d0 + s (d1 + s (d2 + s d3)) with d_k = c_k / dZ^k -- five doubles per interval,
// {Z_m, d0 | d1, d2} as two 128-byte lines of 8 copies (LDS.128, lane l reads copy l & 7) and d3 as one line of
// 16 copies (LDS.64, copy l & 15): 10 conflict-free wavefronts per warp (c0..c3 + {Z, 1/dZ}: 12).
// (the fast path takes its logarithms with ln_tab, pdfb_internal.cuh: the node logarithm stored here
// comes from the same function, so that a query on a node gets s = 0 exactly and returns the node value)
__global__ void k1_alphas_lines(const IntervalRec *__restrict__ rec, const double *__restrict__ a,
                                const double *__restrict__ q2k, unsigned char *__restrict__ lines,
                                const double2 *__restrict__ lntab, int lo, int M)
{
    int m = blockIdx.x * blockDim.x + threadIdx.x;  // interval m of the sub-grid [lo, lo+M)
    if (m >= M) return;
    double d[4] = {0.0, 0.0, 0.0, 0.0};
    const IntervalRec r = rec[lo + m];
    const double q = q2k[lo + m];
    const double z = ln_tab(q, lntab[ln_tab_bin(q) * 8]);
    if (m < M - 1) {
        const double y0 = a[lo + m], y1 = a[lo + m + 1];
        const double ym = a[lo + max(m - 1, 0)], yp = a[lo + min(m + 2, M - 1)];
        const double dL = fma(r.aLm, ym, fma(r.aL0, y0, r.aL1 * y1));
        const double dH = fma(r.aHp, yp, fma(r.aH0, y0, r.aH1 * y1));
        const double dy = y1 - y0;
        d[0] = y0;
        d[1] = dL * r.inv_dz;
        d[2] = (3.0 * dy - 2.0 * dL - dH) * r.inv_dz * r.inv_dz;
        d[3] = (dL + dH - 2.0 * dy) * r.inv_dz * r.inv_dz * r.inv_dz;
    }
    double2 *dst = reinterpret_cast<double2 *>(lines + (size_t)(lo + m) * PDFB_ALPHAS_LINE);
    for (int c = 0; c < 8; c++) { dst[c] = make_double2(z, d[0]); dst[8 + c] = make_double2(d[1], d[2]); dst[16 + c] = make_double2(d[3], d[3]); }
}

int pdfb_setup_alphas_fast(const IntervalRec *d_rec, const double *d_a, const double *d_q2k, unsigned char *d_lines,
                           const double2 *d_lntab, int n_sub, const int *h_off, cudaStream_t st)
{
    for (int s = 0; s < n_sub; s++) {
        int M = h_off[s + 1] - h_off[s];
        k1_alphas_lines<<<(M + 63) / 64, 64, 0, st>>>(d_rec, d_a, d_q2k, d_lines, d_lntab, h_off[s], M);
        pdfb_count_launch(1);
    }
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
