// capi.cu -- the C-ABI of include/pdfb200.h: validation, host grid manager, handles.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "pdfb_internal.cuh"

static std::atomic<long long> g_launches{0};
void pdfb_count_launch(int n) { g_launches += n; }
extern "C" long long pdfb_launch_count(void) { return g_launches.load(); }

extern "C" const char *pdfb_strerror(int code)
{
    switch (code) {
    case PDFB_OK: return "ok";
    case PDFB_EINVAL: return "invalid argument (null pointer, negative size or bad count)";
    case PDFB_EKNOTS: return "bad knots (not increasing, non-positive, sub-grids not sharing their threshold, or < 2 knots)";
    case PDFB_EPID: return "requested PID is not in the grid";
    case PDFB_ECUDA: return "CUDA runtime error (no device, out of memory or launch failure)";
    case PDFB_EIO: return "file could not be opened or read";
    case PDFB_EFORMAT: return "file is not in the expected LHAPDF text layout";
    case PDFB_EXKNOTS: return "sub-grids with different PID lists, or sub-grids with their own x-knot arrays passed to an entry point that takes one array (use pdf_grid_load_xs / pdfb_lhagrid_*_xs)";
    case PDFB_ELIMIT: return "too many sub-grids, PIDs or alpha_s nodes";
    case PDFB_ESTATIC: return "alphas_q2_static takes at most 256 nodes (PDFB_STATIC_MAX_KNOTS): the node table must fit the library's fixed scratch array; load longer lists with alphas_grid_load";
    default: return "unknown pdfb error code";
    }
}

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Search LUT over [Z_0, Z_{nk-1}] (ln knots) for knots 0..kmax with raw values R; the entry
// encoding is described in pdfb_internal.cuh.
void pdfb_fill_lut(unsigned short *lut, const double *Z, const double *R, int nk, int kmax)
{
    const double h = (Z[nk - 1] - Z[0]) / PDFB_LUT_BINS, mg = 1e-6 * h;  // safety margin at bin edges
    for (int b = 0; b < PDFB_LUT_BINS; b++) {
        const double lo = Z[0] + b * h - mg, hi = Z[0] + (b + 1) * h + mg;
        int m0 = 0, first = -1, last = -1, multi = 0;
        for (int k = 1; k <= kmax; k++) {
            if (Z[k] <= lo) m0 = k;
            else if (Z[k] <= hi) {
                if (first < 0) first = k;
                else if (R[k] != R[first]) multi = 1;
                last = k;
            }
        }
        int delta = (first >= 0 && !multi) ? last - m0 : 0;
        if (delta > 3) { multi = 1; delta = 0; }
        lut[b] = (unsigned short)((m0 << 3) | (delta << 1) | multi);
    }
}

// ------------------------------------------------------------------------------ PDF grid
extern "C" int pdf_set_load(int n_members, int n_sub, int nx, const double *x_knots, const int *q_offsets,
                            const double *q_knots, int n_pid, const int *pids, const double *values,
                            int device, pdfb_grid **out)
{
    if (n_members < 1 || n_members > PDFB_MAX_MEMBERS) return out ? (*out = nullptr, PDFB_ELIMIT) : PDFB_EINVAL;
    if (!out) return PDFB_EINVAL;
    *out = nullptr;
    if (!x_knots || !q_offsets || !q_knots || !pids || !values) return PDFB_EINVAL;
    if (n_sub < 1 || nx < 2 || n_pid < 1 || q_offsets[0] != 0) return PDFB_EINVAL;
    if (n_sub > PDFB_MAX_SUBGRIDS || n_pid > PDFB_MAX_PIDS) return PDFB_ELIMIT;
    for (int i = 0; i < nx; i++) {
        if (!(x_knots[i] > 0.0) || !std::isfinite(x_knots[i])) return PDFB_EKNOTS;
        if (i && !(x_knots[i] > x_knots[i - 1])) return PDFB_EKNOTS;
    }
    for (int s = 0; s < n_sub; s++) {
        int a = q_offsets[s], b = q_offsets[s + 1];
        if (b - a < 2) return PDFB_EKNOTS;
        for (int j = a; j < b; j++) {
            if (!(q_knots[j] > 0.0) || !std::isfinite(q_knots[j])) return PDFB_EKNOTS;
            if (j > a && !(q_knots[j] > q_knots[j - 1])) return PDFB_EKNOTS;
        }
        if (s && q_knots[a] != q_knots[a - 1]) return PDFB_EKNOTS;
    }
    const int nq_tot = q_offsets[n_sub];
    {   // table values must be finite: the kernels multiply out-of-stencil knots by weights that are exactly 0
        const long long tot = (long long)n_members * nx * nq_tot * n_pid;
        for (long long e = 0; e < tot; e++) if (!std::isfinite(values[e])) return PDFB_EINVAL;
    }

    if (!(x_knots[0] >= 1e-300) || !(q_knots[0] * q_knots[0] >= 1e-300)) return PDFB_EKNOTS;  // subnormal coordinates

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return PDFB_ECUDA;
    DeviceGuard guard(device);  // the caller's current device is put back on return
    if (!guard.ok) return PDFB_ECUDA;

    pdfb_grid *g = new (std::nothrow) pdfb_grid();
    if (!g) return PDFB_EINVAL;
    g->rr_cap_next.store(0);
    g->rr_next.store(0);  // (new pdfb_grid() value-initialises: every other member is zero)
    g->device = device;
    if (cudaDeviceGetAttribute(&g->sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { delete g; return PDFB_ECUDA; }
    GridDev &d = g->d;
    d.n_sub = n_sub; d.nx = nx; d.n_pid = n_pid; d.nq_tot = nq_tot; d.n_members = n_members;
    d.kpad = (n_pid + 1) & ~1;  // even number of doubles per knot: 16-byte aligned knots
    memcpy(g->pids, pids, sizeof(int) * n_pid);

    // host-side knot arrays: raw and ln
    // (ln knots are computed on the device by K1 with the function the queries use, reading R-ln)
    std::vector<double> h_q2(nq_tot + 1), h_z(nx + nq_tot + 1);
    for (int j = 0; j < nq_tot; j++) h_q2[j] = q_knots[j] * q_knots[j];
    h_q2[nq_tot] = 1.01 * h_q2[0];  // rule C's second probe scale rides along
    long long knots = 0;
    for (int s = 0; s < n_sub; s++) {
        d.q_off[s] = q_offsets[s];
        d.v_off[s] = (int)knots;
        d.q2_lo[s] = h_q2[q_offsets[s]];
        knots += (long long)nx * (q_offsets[s + 1] - q_offsets[s]);
    }
    d.q_off[n_sub] = nq_tot;
    d.x_min = x_knots[0]; d.x_max = x_knots[nx - 1];
    d.q2_min = h_q2[0]; d.q2_max = h_q2[nq_tot - 1];

    // one device blob: [xk | q2k | z (ln knots) | xrec | qrec | val | counter | valg | valg2 | aux | row ranges | lists];
    // the uploaded file-order values live in a staging allocation of their own, freed after K1
    size_t o_xk = 0;
    size_t o_q2k = align_up(o_xk + sizeof(double) * nx, 128);
    size_t o_z = align_up(o_q2k + sizeof(double) * (nq_tot + 1), 128);
    size_t o_xrec = align_up(o_z + sizeof(double) * (nx + nq_tot + 1), 128);
    size_t o_qrec = align_up(o_xrec + sizeof(IntervalRec) * nx, 128);
    size_t o_val = align_up(o_qrec + sizeof(IntervalRec) * nq_tot, 128);
    d.val_mstride = knots * d.kpad;  // one member's table, in doubles
    // shared-memory path: flavour-group slices and the aux block
    d.nx4 = (nx + 3) & ~3;
    d.n_groups = (n_pid + 3) / 4;
    d.slice_bytes = nq_tot * d.nx4 * 32;
    d.nx2 = nx + ((4 - nx % 8) + 8) % 8;  // smallest >= nx that is 4 (mod 8)
    d.n_groups2 = (n_pid + 1) / 2;
    d.slice2_bytes = nq_tot * d.nx2 * 16;
    d.smem_ok = (nx >= 4);
    for (int s = 0; s < n_sub; s++) if (q_offsets[s + 1] - q_offsets[s] < 4) d.smem_ok = 0;
    if (nq_tot >= 8192 || nx >= 8192) d.smem_ok = 0;  // LUT entry bit budget
    d.a_lutx = 0;
    d.a_lutq = d.a_lutx + 2 * PDFB_LUT_BINS;
    d.a_xk = d.a_lutq + 2 * PDFB_LUT_BINS;
    d.a_q2k = d.a_xk + (int)sizeof(double) * nx;
    d.a_xrec = (int)align_up(d.a_q2k + sizeof(double) * nq_tot, 128);
    d.pre_bytes = d.a_xrec + 128 * nx;            // the slice starts here, 128-byte aligned
    d.a_qrec = 0;
    // a stencil may reach two rows plus three knots past the table (the phantom interval of the last Q^2
    // knot, xfxq2_smem.cuh): keep that much finite data there
    d.post_bytes = (int)align_up((size_t)std::max(128 * nq_tot, 2 * d.nx4 * 32 + 128), 128);
    if (128 * nx < d.nx4 * 32 + 32) d.smem_ok = 0;  // (never: 128 nx >= 32 nx4 + 32 for nx >= 2)
    const int aux_bytes = d.pre_bytes + d.post_bytes;
    // which layouts this handle will ever read (a set of 400 members is ~1 GB if all are kept):
    // the shared-memory path takes the 4-column slices (bit 0) and / or the 2-column slices (bit 1);
    // the [iq][ix][kpad] table serves the read-only-cache kernel -- every member if that kernel is the
    // only path, else member 0 alone (the general kernel of pdf_lumi_events)
    if (d.smem_ok) d.smem_ok = pdfb_smem_eligible(g);
    const int n_val = d.smem_ok ? 1 : n_members;
    const int n_g4 = (d.smem_ok & 1) ? n_members : 0, n_g2 = (d.smem_ok & 2) ? n_members : 0;
    size_t o_cnt = align_up(o_val + sizeof(double) * knots * d.kpad * n_val, 128);
    size_t o_valg = align_up(o_cnt + 128, 128);
    size_t o_valg2 = align_up(o_valg + (size_t)d.slice_bytes * d.n_groups * n_g4, 128);
    size_t o_aux = align_up(o_valg2 + (size_t)d.slice2_bytes * d.n_groups2 * n_g2, 128);
    size_t o_rr = align_up(o_aux + aux_bytes, 128);
    size_t o_ws = align_up(o_rr + sizeof(int) * 2 * (PDFB_RR_SLOTS + PDFB_RR_CAP_SLOTS), 128);
    size_t total = o_ws + PDFB_WS_BYTES;
    char *blob = nullptr, *raw = nullptr;
    const long long member_values = knots * n_pid;  // doubles of one member in file order
    if (cudaMalloc(&blob, total) != cudaSuccess) { delete g; return PDFB_ECUDA; }
    if (cudaMalloc(&raw, sizeof(double) * member_values * n_members) != cudaSuccess) { cudaFree(blob); delete g; return PDFB_ECUDA; }
    g->blob = blob; g->blob_bytes = total;

    int rc = PDFB_OK;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        if (e0) cudaEventDestroy(e0);
        cudaFree(raw); cudaFree(blob); delete g;
        return PDFB_ECUDA;
    }
    do {
        if (cudaMemcpy(blob + o_xk, x_knots, sizeof(double) * nx, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(blob + o_q2k, h_q2.data(), sizeof(double) * (nq_tot + 1), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(raw, values, sizeof(double) * member_values * n_members, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemset(blob + o_cnt, 0, 128) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        cudaEventRecord(e0, 0);
        // K1: ln of the knots (and of rule C's probe scale), read back for the host-side tables
        rc = pdfb_setup_ln((const double *)(blob + o_xk), (double *)(blob + o_z), nx, 0);
        if (!rc) rc = pdfb_setup_ln((const double *)(blob + o_q2k), (double *)(blob + o_z) + nx, nq_tot + 1, 0);
        if (rc) break;
        if (cudaMemcpy(h_z.data(), blob + o_z, sizeof(double) * (nx + nq_tot + 1), cudaMemcpyDeviceToHost) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        d.U0 = h_z[0]; d.U1 = h_z[1]; d.inv_dU01 = 1.0 / (h_z[1] - h_z[0]);
        d.Va = h_z[nx + nq_tot - 2]; d.Vb = h_z[nx + nq_tot - 1]; d.inv_dVab = 1.0 / (d.Vb - d.Va);
        // K1: interval records for the x knots and for each sub-grid's Q^2 knots
        int xoff[2] = {0, nx};
        {   // host part of the aux block: raw knots, search LUTs, sub-grid of each Q^2 knot
            std::vector<unsigned char> aux(aux_bytes, 0);
            memcpy(aux.data() + d.a_xk, x_knots, sizeof(double) * nx);
            memcpy(aux.data() + d.a_q2k, h_q2.data(), sizeof(double) * nq_tot);
            unsigned short *lx = (unsigned short *)(aux.data() + d.a_lutx);
            unsigned short *lq = (unsigned short *)(aux.data() + d.a_lutq);
            const double *U = h_z.data(), *V = h_z.data() + nx;
            d.lutx_u0 = U[0]; d.lutx_inv_h = PDFB_LUT_BINS / (U[nx - 1] - U[0]);
            d.lutq_v0 = V[0]; d.lutq_inv_h = PDFB_LUT_BINS / (V[nq_tot - 1] - V[0]);
            pdfb_fill_lut(lx, U, x_knots, nx, nx - 1);          // (the last knot starts its phantom interval, xfxq2_smem.cuh)
            pdfb_fill_lut(lq, V, h_q2.data(), nq_tot, nq_tot - 1);  // concatenated Q^2 knots
            if (cudaMemcpy(blob + o_aux, aux.data(), aux_bytes, cudaMemcpyHostToDevice) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        }
        rc = pdfb_setup_records((const double *)(blob + o_z), (IntervalRec *)(blob + o_xrec),
                                (IntervalRec32 *)(blob + o_aux + d.a_xrec), 1, xoff, 0);
        if (rc) break;
        rc = pdfb_setup_records((const double *)(blob + o_z) + nx, (IntervalRec *)(blob + o_qrec),
                                (IntervalRec32 *)(blob + o_aux + d.pre_bytes + d.a_qrec), n_sub, d.q_off, 0);
        if (rc) break;
        // K1: value table re-layout, sub-grid by sub-grid, all members of a layout in one launch
        long long src = 0;
        for (int s = 0; s < n_sub && !rc; s++) {
            int nq = q_offsets[s + 1] - q_offsets[s];
            rc = pdfb_setup_values((const double *)raw + src, (double *)(blob + o_val) + (long long)d.v_off[s] * d.kpad,
                                   nx, nq, n_pid, d.kpad, 0, n_val, member_values, d.val_mstride);
            if (!rc && n_g4) rc = pdfb_setup_group_slices((const double *)raw + src, (double *)(blob + o_valg),
                                                          q_offsets[s] * d.nx4, nx, d.nx4, nq, n_pid, d.n_groups,
                                                          (long long)d.slice_bytes / 8, 0, 4, n_g4, member_values);
            if (!rc && n_g2) rc = pdfb_setup_group_slices((const double *)raw + src, (double *)(blob + o_valg2),
                                                          q_offsets[s] * d.nx2, nx, d.nx2, nq, n_pid, d.n_groups2,
                                                          (long long)d.slice2_bytes / 8, 0, 2, n_g2, member_values);
            src += (long long)nx * nq * n_pid;
        }
        if (rc) break;
        cudaEventRecord(e1, 0);
        if (cudaDeviceSynchronize() != cudaSuccess) { rc = PDFB_ECUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        g->setup_ms = ms;
        // rule C's second probe sits at the fixed scale 1.01 * q2_min: its v weights are constants
        double qC = h_q2[nq_tot];
        int nq0 = q_offsets[1];
        if (!(qC < h_q2[nq0 - 1])) { rc = PDFB_EKNOTS; break; }
        int jC = 0;
        for (int m = 1; m <= nq0 - 2; m++) if (h_q2[m] <= qC) jC = m;
        IntervalRec rC;
        if (cudaMemcpy(&rC, blob + o_qrec + sizeof(IntervalRec) * jC, sizeof(rC), cudaMemcpyDeviceToHost) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        d.jC = jC;
        weights4(rC, (h_z[nx + nq_tot] - rC.z0) * rC.inv_dz, d.wvC);
    } while (0);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(raw);  // (the device is idle: synchronised above, or setup failed)
    if (rc) { cudaFree(blob); delete g; return rc; }

    d.xk = (const double *)(blob + o_xk);
    d.q2k = (const double *)(blob + o_q2k);
    d.xrec = (const IntervalRec *)(blob + o_xrec);
    d.qrec = (const IntervalRec *)(blob + o_qrec);
    d.val = (const double *)(blob + o_val);
    d.n_invalid = (unsigned long long *)(blob + o_cnt);
    d.valg = (const double *)(blob + o_valg);
    d.valg2 = (const double *)(blob + o_valg2);
    d.aux = (const unsigned char *)(blob + o_aux);
    d.slow_ws = (uint32_t *)(blob + o_ws);
    d.row_range = (int *)(blob + o_rr);
    pdfb_lumi_plan(g);
    *out = g;
    return PDFB_OK;
}

static int resolve_cols(const pdfb_grid *g, int n_req, const int *pids, int *cols)
{
    if (n_req < 1 || n_req > PDFB_MAX_PIDS) return PDFB_EINVAL;
    for (int r = 0; r < n_req; r++) {
        int pid = pids[r] == 0 ? 21 : pids[r];
        cols[r] = -1;
        for (int k = 0; k < g->d.n_pid; k++) if (g->pids[k] == pid) cols[r] = k;
        if (cols[r] < 0) return PDFB_EPID;
    }
    return PDFB_OK;
}

extern "C" int pdf_grid_load(int n_sub, int nx, const double *x_knots, const int *q_offsets,
                             const double *q_knots, int n_pid, const int *pids, const double *values,
                             int device, pdfb_grid **out)
{
    return pdf_set_load(1, n_sub, nx, x_knots, q_offsets, q_knots, n_pid, pids, values, device, out);
}

extern "C" int pdf_set_members(const pdfb_grid *g) { return g ? g->d.n_members : 0; }

static int members_impl(const pdfb_grid *g, int member0, int n_mem, int n_req, const int *pids, long long n,
                        const double *x, const double *q2, double *out, void *cuda_stream, int q_is_q)
{
    if (!g || !pids || n < 0 || n_mem < 0) return PDFB_EINVAL;
    if (member0 < 0 || member0 + n_mem > g->d.n_members) return PDFB_EINVAL;
    if (n > 0 && n_mem > 0 && (!x || !q2 || !out)) return PDFB_EINVAL;
    int cols[PDFB_MAX_PIDS];
    int rc = resolve_cols(g, n_req, pids, cols);
    if (rc) return rc;
    if (n_mem == 0) return PDFB_OK;
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    return pdfb_launch_xfxq2(g, n_req, cols, n, x, q2, out, n, (cudaStream_t)cuda_stream, q_is_q, member0, n_mem);
}

extern "C" int pdf_xfxq2_members(const pdfb_grid *g, int member0, int n_mem, int n_req, const int *pids,
                                 long long n, const double *x, const double *q2, double *out, void *cuda_stream)
{
    return members_impl(g, member0, n_mem, n_req, pids, n, x, q2, out, cuda_stream, 0);
}

extern "C" int pdf_xfxq_members(const pdfb_grid *g, int member0, int n_mem, int n_req, const int *pids,
                                long long n, const double *x, const double *q, double *out, void *cuda_stream)
{
    return members_impl(g, member0, n_mem, n_req, pids, n, x, q, out, cuda_stream, 1);
}

extern "C" int pdf_xfxq2(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                         const double *q2, double *out, void *cuda_stream)
{
    if (!g || !pids || n < 0) return PDFB_EINVAL;
    if (n > 0 && (!x || !q2 || !out)) return PDFB_EINVAL;
    int cols[PDFB_MAX_PIDS];
    int rc = resolve_cols(g, n_req, pids, cols);
    if (rc) return rc;
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    return pdfb_launch_xfxq2(g, n_req, cols, n, x, q2, out, n, (cudaStream_t)cuda_stream);
}

// the two layout / precision variants of pdf_xfxq2 (compile-time kernel variants)
static int xfxq2_variant(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x, const double *q2,
                         void *out, void *cuda_stream, int mode)
{
    if (!g || !pids || n < 0) return PDFB_EINVAL;
    if (n > 0 && (!x || !q2 || !out)) return PDFB_EINVAL;
    int cols[PDFB_MAX_PIDS];
    int rc = resolve_cols(g, n_req, pids, cols);
    if (rc) return rc;
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    return pdfb_launch_xfxq2(g, n_req, cols, n, x, q2, (double *)out, n, (cudaStream_t)cuda_stream, mode);
}

extern "C" int pdf_xfxq2_pm(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                            const double *q2, double *out, void *cuda_stream)
{
    return xfxq2_variant(g, n_req, pids, n, x, q2, out, cuda_stream, 1 << 1);
}

extern "C" int pdf_xfxq2_f32(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                             const double *q2, float *out, void *cuda_stream)
{
    return xfxq2_variant(g, n_req, pids, n, x, q2, out, cuda_stream, 2 << 1);
}

extern "C" int pdf_xfxq(const pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                        const double *q, double *out, void *cuda_stream)
{
    if (!g || !pids || n < 0) return PDFB_EINVAL;
    if (n > 0 && (!x || !q || !out)) return PDFB_EINVAL;
    int cols[PDFB_MAX_PIDS];
    int rc = resolve_cols(g, n_req, pids, cols);
    if (rc) return rc;
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    return pdfb_launch_xfxq2(g, n_req, cols, n, x, q, out, n, (cudaStream_t)cuda_stream, 1);
}

extern "C" int pdf_grid_uses_smem_path(const pdfb_grid *g) { return g ? (g->d.smem_ok != 0) : 0; }

extern "C" int pdf_grid_status(const pdfb_grid *g, long long *n_invalid_points)
{
    if (!g || !n_invalid_points) return PDFB_EINVAL;
    unsigned long long c = 0;
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    PDFB_CUDA(cudaDeviceSynchronize());
    PDFB_CUDA(cudaMemcpy(&c, g->d.n_invalid, sizeof(c), cudaMemcpyDeviceToHost));
    *n_invalid_points = (long long)c;
    return PDFB_OK;
}

extern "C" void pdf_grid_free(pdfb_grid *g)
{
    if (!g) return;
    DeviceGuard guard(g->device);
    cudaDeviceSynchronize();
    for (int i = 0; i < 3; i++)
        if (g->streams[i]) cudaStreamDestroy(g->streams[i]);
    if (g->stage) cudaFree(g->stage);
    if (g->blob) cudaFree(g->blob);
    delete g;
}
