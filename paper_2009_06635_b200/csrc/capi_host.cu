// capi_host.cu -- alpha_s handle management and the HOST-buffer entry points
// (pdf_xfxq2_host, alphas_q2_host): chunked copy-in / evaluate / copy-out pipelines.
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "pdfb_internal.cuh"

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

extern "C" double pdf_grid_setup_ms(const pdfb_grid *g) { return g ? g->setup_ms : -1.0; }

// ------------------------------------------------------------------------------ alpha_s
extern "C" int alphas_grid_load(int n_knots, const double *q_knots, const double *alphas, int device,
                                pdfb_alphas **out)
{
    if (!out) return PDFB_EINVAL;
    *out = nullptr;
    if (!q_knots || !alphas || n_knots < 2) return PDFB_EINVAL;
    if (n_knots > 512) return PDFB_ELIMIT;
    std::vector<int> off(1, 0);
    for (int k = 0; k < n_knots; k++) {
        if (!(q_knots[k] > 0.0) || !std::isfinite(q_knots[k]) || !std::isfinite(alphas[k])) return PDFB_EKNOTS;
        if (k && q_knots[k] < q_knots[k - 1]) return PDFB_EKNOTS;
        if (k && q_knots[k] == q_knots[k - 1]) off.push_back(k);
    }
    off.push_back(n_knots);
    int n_sub = (int)off.size() - 1;
    if (n_sub > PDFB_MAX_SUBGRIDS) return PDFB_ELIMIT;
    for (int s = 0; s < n_sub; s++) if (off[s + 1] - off[s] < 2) return PDFB_EKNOTS;

    if (!(q_knots[0] * q_knots[0] >= 1e-300)) return PDFB_EKNOTS;  // subnormal scale

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return PDFB_ECUDA;
    DeviceGuard guard(device);
    if (!guard.ok) return PDFB_ECUDA;
    pdfb_alphas *a = new (std::nothrow) pdfb_alphas();
    if (!a) return PDFB_EINVAL;
    memset(a, 0, sizeof(*a));
    a->device = device;
    if (cudaDeviceGetAttribute(&a->sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) { delete a; return PDFB_ECUDA; }
    AlphasDev &d = a->d;
    d.K = n_knots; d.n_sub = n_sub;
    std::vector<double> h_q2(n_knots), h_z(n_knots);
    for (int k = 0; k < n_knots; k++) h_q2[k] = q_knots[k] * q_knots[k];
    for (int s = 0; s <= n_sub; s++) d.off[s] = off[s];
    for (int s = 0; s < n_sub; s++) d.q2_lo[s] = h_q2[off[s]];
    d.q2_min = h_q2[0]; d.q2_max = h_q2[n_knots - 1];
    d.a_first = alphas[0]; d.a_last = alphas[n_knots - 1];

    size_t o_q2 = 0, o_a = align_up(sizeof(double) * n_knots, 128), o_z = 2 * o_a, o_rec = 3 * o_a;
    // fast-path block: [lines K*384][ln table][q2k K doubles][lut u16]
    d.fast_ok = (n_knots <= 192);
    d.f_lntab = PDFB_ALPHAS_LINE * n_knots;
    d.f_q2k = d.f_lntab + PDFB_LNTAB_BYTES;
    d.f_lut = d.f_q2k + (int)sizeof(double) * n_knots;
    d.fast_bytes = (int)align_up(d.f_lut + 2 * PDFB_LUT_BINS, 16);
    size_t o_fast = align_up(o_rec + sizeof(IntervalRec) * n_knots, 128);
    size_t total = o_fast + d.fast_bytes;
    char *blob = nullptr;
    if (cudaMalloc(&blob, total) != cudaSuccess) { delete a; return PDFB_ECUDA; }
    a->blob = blob;
    int rc = PDFB_OK;
    if (cudaMemcpy(blob + o_q2, h_q2.data(), sizeof(double) * n_knots, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(blob + o_a, alphas, sizeof(double) * n_knots, cudaMemcpyHostToDevice) != cudaSuccess)
        rc = PDFB_ECUDA;
    if (!rc) rc = pdfb_setup_ln((const double *)(blob + o_q2), (double *)(blob + o_z), n_knots, 0);
    if (!rc) rc = pdfb_setup_records((const double *)(blob + o_z), (IntervalRec *)(blob + o_rec), nullptr, n_sub, d.off, 0);
    if (!rc) {  // ln table of the fast path: entry j = {1/c_j, ln c_j}, c_j = 1 + (j + 1/2)/64, 8 copies per line
        std::vector<double> tab(PDFB_LNTAB_BYTES / 8);
        for (int j = 0; j < 64; j++) {
            const double c = 1.0 + (j + 0.5) / 64.0;
            for (int k = 0; k < 8; k++) { tab[(j * 8 + k) * 2] = 1.0 / c; tab[(j * 8 + k) * 2 + 1] = std::log(c); }
        }
        if (cudaMemcpy(blob + o_fast + d.f_lntab, tab.data(), PDFB_LNTAB_BYTES, cudaMemcpyHostToDevice) != cudaSuccess) rc = PDFB_ECUDA;
    }
    if (!rc) rc = pdfb_setup_alphas_fast((const IntervalRec *)(blob + o_rec), (const double *)(blob + o_a),
                                         (const double *)(blob + o_q2), (unsigned char *)(blob + o_fast),
                                         (const double2 *)(blob + o_fast + d.f_lntab), n_sub, d.off, 0);
    if (!rc && cudaMemcpy(h_z.data(), blob + o_z, sizeof(double) * n_knots, cudaMemcpyDeviceToHost) != cudaSuccess) rc = PDFB_ECUDA;
    if (!rc) {  // LUT over ln Q^2 (encoding in pdfb_internal.cuh); a repeated node lands on its upper copy
        std::vector<unsigned short> lut(PDFB_LUT_BINS);
        d.lut_v0 = h_z[0]; d.lut_inv_h = PDFB_LUT_BINS / (h_z[n_knots - 1] - h_z[0]);
        pdfb_fill_lut(lut.data(), h_z.data(), h_q2.data(), n_knots, n_knots - 1);
        if (cudaMemcpy(blob + o_fast + d.f_q2k, h_q2.data(), sizeof(double) * n_knots, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(blob + o_fast + d.f_lut, lut.data(), 2 * PDFB_LUT_BINS, cudaMemcpyHostToDevice) != cudaSuccess)
            rc = PDFB_ECUDA;
    }
    if (!rc && cudaDeviceSynchronize() != cudaSuccess) rc = PDFB_ECUDA;
    if (rc) { cudaFree(blob); delete a; return rc; }
    d.fast = (const unsigned char *)(blob + o_fast);
    d.q2k = (const double *)(blob + o_q2);
    d.a = (const double *)(blob + o_a);
    d.rec = (const IntervalRec *)(blob + o_rec);
    *out = a;
    return PDFB_OK;
}

extern "C" int alphas_q2(const pdfb_alphas *a, long long n, const double *q2, double *out, void *cuda_stream)
{
    if (!a || n < 0) return PDFB_EINVAL;
    if (n > 0 && (!q2 || !out)) return PDFB_EINVAL;
    DeviceGuard guard(a->device);
    if (!guard.ok) return PDFB_ECUDA;
    return pdfb_launch_alphas(a, n, q2, out, (cudaStream_t)cuda_stream);
}

extern "C" int alphas_q(const pdfb_alphas *a, long long n, const double *q, double *out, void *cuda_stream)
{
    if (!a || n < 0) return PDFB_EINVAL;
    if (n > 0 && (!q || !out)) return PDFB_EINVAL;
    DeviceGuard guard(a->device);
    if (!guard.ok) return PDFB_ECUDA;
    return pdfb_launch_alphas(a, n, q, out, (cudaStream_t)cuda_stream, 1);
}

extern "C" void alphas_grid_free(pdfb_alphas *a)
{
    if (!a) return;
    DeviceGuard guard(a->device);
    cudaDeviceSynchronize();
    for (int i = 0; i < 2; i++) if (a->streams[i]) cudaStreamDestroy(a->streams[i]);
    if (a->stage) cudaFree(a->stage);
    if (a->blob) cudaFree(a->blob);
    delete a;
}

// ------------------------------------------------------------------------------ host pipelines
static const long long HOST_CHUNK = 1LL << 22;  // points per pipeline stage (32 MiB per input array)

extern "C" int pdf_xfxq2_host(pdfb_grid *g, int n_req, const int *pids, long long n, const double *x,
                              const double *q2, double *out)
{
    if (!g || !pids || n < 0) return PDFB_EINVAL;
    if (n == 0) return PDFB_OK;
    if (!x || !q2 || !out) return PDFB_EINVAL;
    int cols[PDFB_MAX_PIDS];
    if (n_req < 1 || n_req > PDFB_MAX_PIDS) return PDFB_EINVAL;
    for (int r = 0; r < n_req; r++) {
        int pid = pids[r] == 0 ? 21 : pids[r];
        cols[r] = -1;
        for (int k = 0; k < g->d.n_pid; k++) if (g->pids[k] == pid) cols[r] = k;
        if (cols[r] < 0) return PDFB_EPID;
    }
    DeviceGuard guard(g->device);
    if (!guard.ok) return PDFB_ECUDA;
    const int NS = 3;
    const long long chunk = n < HOST_CHUNK ? n : HOST_CHUNK;
    const size_t per_stage = sizeof(double) * chunk * (2 + (size_t)n_req);
    if (g->stage_bytes < per_stage * NS) {
        if (g->stage) cudaFree(g->stage);
        g->stage = nullptr; g->stage_bytes = 0;
        PDFB_CUDA(cudaMalloc(&g->stage, per_stage * NS));
        g->stage_bytes = per_stage * NS;
    }
    for (int i = 0; i < NS; i++) {
        if (!g->streams[i]) PDFB_CUDA(cudaStreamCreateWithFlags(&g->streams[i], cudaStreamNonBlocking));
    }
    int rc = PDFB_OK;
    int stage = 0;
    for (long long a = 0; a < n && !rc; a += chunk, stage = (stage + 1) % NS) {
        long long m = (n - a < chunk) ? (n - a) : chunk;
        cudaStream_t st = g->streams[stage];
        double *dx = (double *)((char *)g->stage + per_stage * stage);
        double *dq = dx + chunk, *dout = dq + chunk;
        // stream order serialises reuse of this stage's buffers
        if (cudaMemcpyAsync(dx, x + a, sizeof(double) * m, cudaMemcpyHostToDevice, st) != cudaSuccess ||
            cudaMemcpyAsync(dq, q2 + a, sizeof(double) * m, cudaMemcpyHostToDevice, st) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        rc = pdfb_launch_xfxq2(g, n_req, cols, m, dx, dq, dout, chunk, st);
        if (rc) break;
        // one copy per flavour row (a 2-D copy would cap the pitch 8 n at cudaDevAttrMaxPitch: n < 2^28)
        for (int r = 0; r < n_req && !rc; r++)
            if (cudaMemcpyAsync(out + (size_t)r * n + a, dout + (size_t)r * chunk, sizeof(double) * m, cudaMemcpyDeviceToHost, st) != cudaSuccess)
                rc = PDFB_ECUDA;
    }
    for (int i = 0; i < NS; i++) if (cudaStreamSynchronize(g->streams[i]) != cudaSuccess) rc = rc ? rc : PDFB_ECUDA;
    return rc;
}

extern "C" int alphas_q2_host(pdfb_alphas *a, long long n, const double *q2, double *out)
{
    if (!a || n < 0) return PDFB_EINVAL;
    if (n == 0) return PDFB_OK;
    if (!q2 || !out) return PDFB_EINVAL;
    DeviceGuard guard(a->device);
    if (!guard.ok) return PDFB_ECUDA;
    const int NS = 2;
    const long long chunk = n < HOST_CHUNK ? n : HOST_CHUNK;
    const size_t per_stage = sizeof(double) * chunk * 2;
    if (a->stage_bytes < per_stage * NS) {
        if (a->stage) cudaFree(a->stage);
        a->stage = nullptr; a->stage_bytes = 0;
        PDFB_CUDA(cudaMalloc(&a->stage, per_stage * NS));
        a->stage_bytes = per_stage * NS;
    }
    for (int i = 0; i < NS; i++)
        if (!a->streams[i]) PDFB_CUDA(cudaStreamCreateWithFlags(&a->streams[i], cudaStreamNonBlocking));
    int rc = PDFB_OK, stage = 0;
    for (long long b = 0; b < n && !rc; b += chunk, stage = (stage + 1) % NS) {
        long long m = (n - b < chunk) ? (n - b) : chunk;
        cudaStream_t st = a->streams[stage];
        double *dq = (double *)((char *)a->stage + per_stage * stage), *dout = dq + chunk;
        if (cudaMemcpyAsync(dq, q2 + b, sizeof(double) * m, cudaMemcpyHostToDevice, st) != cudaSuccess) { rc = PDFB_ECUDA; break; }
        rc = pdfb_launch_alphas(a, m, dq, dout, st);
        if (rc) break;
        if (cudaMemcpyAsync(out + b, dout, sizeof(double) * m, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = PDFB_ECUDA;
    }
    for (int i = 0; i < NS; i++) if (cudaStreamSynchronize(a->streams[i]) != cudaSuccess) rc = rc ? rc : PDFB_ECUDA;
    return rc;
}
