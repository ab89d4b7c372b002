// capi_xs.cu -- pdf_grid_load_xs: a PDF member whose sub-grids carry their OWN x-knot arrays, as the
// LHAPDF6 grid layout allows (every sub-grid block of a member file has its own x line; PAPER.md:67:
// the files "are directly loaded", sub-grids are interpolated independently).  Reading:
// the cell, t and the x derivatives of a point come from the x knots of the point's own sub-grid,
// rule A continues from that sub-grid's first two knots.
// Such a grid is evaluated by the read-only-cache kernel (xfxq2_v0.cuh) -- the shared-memory kernel's
// slices, records and search tables assume one x-knot array.  If all arrays are in fact the same, the
// handle is an ordinary pdf_grid_load handle.
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "pdfb_internal.cuh"

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

extern "C" int pdf_grid_load_xs(int n_sub, const int *x_offsets, const double *x_knots, const int *q_offsets,
                                const double *q_knots, int n_pid, const int *pids, const double *values,
                                int device, pdfb_grid **out)
{
    if (!out) return PDFB_EINVAL;
    *out = nullptr;
    if (!x_offsets || !x_knots || !q_offsets || !q_knots || !pids || !values) return PDFB_EINVAL;
    if (n_sub < 1 || n_pid < 1 || q_offsets[0] != 0 || x_offsets[0] != 0) return PDFB_EINVAL;
    if (n_sub > PDFB_MAX_SUBGRIDS || n_pid > PDFB_MAX_PIDS) return PDFB_ELIMIT;
    bool same = true;
    const int nx0 = x_offsets[1];
    for (int s = 0; s < n_sub; s++) {
        const int a = x_offsets[s], b = x_offsets[s + 1];
        if (b - a < 2) return PDFB_EKNOTS;
        for (int i = a; i < b; i++) {
            if (!(x_knots[i] > 0.0) || !std::isfinite(x_knots[i])) return PDFB_EKNOTS;
            if (i > a && !(x_knots[i] > x_knots[i - 1])) return PDFB_EKNOTS;
        }
        // all sub-grids span the same x range (one x_min and x_max for the whole member)
        if (x_knots[a] != x_knots[0] || x_knots[b - 1] != x_knots[nx0 - 1]) return PDFB_EKNOTS;
        if (b - a != nx0 || memcmp(x_knots + a, x_knots, sizeof(double) * nx0)) same = false;
    }
    if (same) return pdf_grid_load(n_sub, nx0, x_knots, q_offsets, q_knots, n_pid, pids, values, device, out);
    for (int s = 0; s < n_sub; s++) {
        const int a = q_offsets[s], b = q_offsets[s + 1];
        if (b - a < 2) return PDFB_EKNOTS;
        for (int j = a; j < b; j++) {
            if (!(q_knots[j] > 0.0) || !std::isfinite(q_knots[j])) return PDFB_EKNOTS;
            if (j > a && !(q_knots[j] > q_knots[j - 1])) return PDFB_EKNOTS;
        }
        if (s && q_knots[a] != q_knots[a - 1]) return PDFB_EKNOTS;
    }
    const int nq_tot = q_offsets[n_sub], nxt = x_offsets[n_sub];
    long long knots = 0;
    for (int s = 0; s < n_sub; s++) knots += (long long)(x_offsets[s + 1] - x_offsets[s]) * (q_offsets[s + 1] - q_offsets[s]);
    for (long long e = 0; e < knots * n_pid; e++) if (!std::isfinite(values[e])) return PDFB_EINVAL;
    if (!(x_knots[0] >= 1e-300) || !(q_knots[0] * q_knots[0] >= 1e-300)) return PDFB_EKNOTS;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return PDFB_ECUDA;
    DeviceGuard guard(device);
    if (!guard.ok) return PDFB_ECUDA;
    pdfb_grid *g = new (std::nothrow) pdfb_grid();
    if (!g) return PDFB_EINVAL;
    g->rr_cap_next.store(0);
    g->rr_next.store(0);  // (new pdfb_grid() value-initialises: every other member is zero)
    g->device = device;
    if (cudaDeviceGetAttribute(&g->sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { delete g; return PDFB_ECUDA; }
    GridDev &d = g->d;
    d.n_sub = n_sub; d.nx = nxt; d.n_pid = n_pid; d.nq_tot = nq_tot; d.n_members = 1;
    d.kpad = (n_pid + 1) & ~1;
    d.xs_per_sub = 1;
    memcpy(g->pids, pids, sizeof(int) * n_pid);
    std::vector<double> h_q2(nq_tot + 1), h_z(nxt + nq_tot + 1);
    for (int j = 0; j < nq_tot; j++) h_q2[j] = q_knots[j] * q_knots[j];
    h_q2[nq_tot] = 1.01 * h_q2[0];  // rule C's second probe scale rides along
    long long kn = 0;
    for (int s = 0; s < n_sub; s++) {
        d.q_off[s] = q_offsets[s]; d.x_off[s] = x_offsets[s];
        d.v_off[s] = (int)kn;
        d.q2_lo[s] = h_q2[q_offsets[s]];
        kn += (long long)(x_offsets[s + 1] - x_offsets[s]) * (q_offsets[s + 1] - q_offsets[s]);
    }
    d.q_off[n_sub] = nq_tot; d.x_off[n_sub] = nxt;
    d.x_min = x_knots[0]; d.x_max = x_knots[nx0 - 1];
    d.q2_min = h_q2[0]; d.q2_max = h_q2[nq_tot - 1];
    d.val_mstride = knots * d.kpad;

    size_t o_xk = 0;
    size_t o_q2k = align_up(o_xk + sizeof(double) * nxt, 128);
    size_t o_z = align_up(o_q2k + sizeof(double) * (nq_tot + 1), 128);
    size_t o_xrec = align_up(o_z + sizeof(double) * (nxt + nq_tot + 1), 128);
    size_t o_qrec = align_up(o_xrec + sizeof(IntervalRec) * nxt, 128);
    size_t o_val = align_up(o_qrec + sizeof(IntervalRec) * nq_tot, 128);
    size_t o_cnt = align_up(o_val + sizeof(double) * knots * d.kpad, 128);
    size_t total = o_cnt + 128;
    char *blob = nullptr, *raw = nullptr;
    if (cudaMalloc(&blob, total) != cudaSuccess) { delete g; return PDFB_ECUDA; }
    if (cudaMalloc(&raw, sizeof(double) * knots * n_pid) != cudaSuccess) { cudaFree(blob); delete g; return PDFB_ECUDA; }
    g->blob = blob; g->blob_bytes = total;
    int rc = PDFB_OK;
    do {
        if (cudaMemcpy(blob + o_xk, x_knots, sizeof(double) * nxt, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(blob + o_q2k, h_q2.data(), sizeof(double) * (nq_tot + 1), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(raw, values, sizeof(double) * knots * n_pid, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemset(blob + o_cnt, 0, 128) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        // K1: ln knots with the queries' own function, interval records per sub-grid array, value re-layout
        rc = pdfb_setup_ln((const double *)(blob + o_xk), (double *)(blob + o_z), nxt, 0);
        if (!rc) rc = pdfb_setup_ln((const double *)(blob + o_q2k), (double *)(blob + o_z) + nxt, nq_tot + 1, 0);
        if (!rc) rc = pdfb_setup_records((const double *)(blob + o_z), (IntervalRec *)(blob + o_xrec), nullptr, n_sub, d.x_off, 0);
        if (!rc) rc = pdfb_setup_records((const double *)(blob + o_z) + nxt, (IntervalRec *)(blob + o_qrec), nullptr, n_sub, d.q_off, 0);
        long long src = 0;
        for (int s = 0; s < n_sub && !rc; s++) {
            const int nxs = x_offsets[s + 1] - x_offsets[s], nq = q_offsets[s + 1] - q_offsets[s];
            rc = pdfb_setup_values((const double *)raw + src, (double *)(blob + o_val) + (long long)d.v_off[s] * d.kpad,
                                   nxs, nq, n_pid, d.kpad, 0, 1, 0, 0);
            src += (long long)nxs * nq * n_pid;
        }
        if (rc) break;
        if (cudaDeviceSynchronize() != cudaSuccess) { rc = PDFB_ECUDA; break; }
        if (cudaMemcpy(h_z.data(), blob + o_z, sizeof(double) * (nxt + nq_tot + 1), cudaMemcpyDeviceToHost) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        d.U0 = h_z[0]; d.U1 = h_z[1]; d.inv_dU01 = 1.0 / (h_z[1] - h_z[0]);
        for (int s = 0; s < n_sub; s++) d.inv_dU01s[s] = 1.0 / (h_z[x_offsets[s] + 1] - h_z[x_offsets[s]]);
        d.Va = h_z[nxt + nq_tot - 2]; d.Vb = h_z[nxt + nq_tot - 1]; d.inv_dVab = 1.0 / (d.Vb - d.Va);
        const double qC = h_q2[nq_tot];
        const int nq0 = q_offsets[1];
        if (!(qC < h_q2[nq0 - 1])) { rc = PDFB_EKNOTS; break; }
        int jC = 0;
        for (int m = 1; m <= nq0 - 2; m++) if (h_q2[m] <= qC) jC = m;
        IntervalRec rC;
        if (cudaMemcpy(&rC, blob + o_qrec + sizeof(IntervalRec) * jC, sizeof(rC), cudaMemcpyDeviceToHost) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        d.jC = jC;
        weights4(rC, (h_z[nxt + nq_tot] - rC.z0) * rC.inv_dz, d.wvC);
    } while (0);
    cudaFree(raw);
    if (rc) { cudaFree(blob); delete g; return rc; }
    d.xk = (const double *)(blob + o_xk);
    d.q2k = (const double *)(blob + o_q2k);
    d.xrec = (const IntervalRec *)(blob + o_xrec);
    d.qrec = (const IntervalRec *)(blob + o_qrec);
    d.val = (const double *)(blob + o_val);
    d.n_invalid = (unsigned long long *)(blob + o_cnt);
    d.smem_ok = 0;      // read-only-cache kernel
    g->lumi_npair = 0;  // pdf_lumi_events: general kernel
    *out = g;
    return PDFB_OK;
}
