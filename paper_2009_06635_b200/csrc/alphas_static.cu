// alphas_static.cu -- alphas_q2_static: alpha_s(Q^2) for callers that must not allocate device memory.
//
// Who that is: PDFFlow lives inside a TensorFlow process, and TensorFlow -- like the
// other frameworks with a caching allocator -- takes nearly all of the GPU's memory for its own pool
// when it starts.  A side library's cudaMalloc in such a process fails with "out of memory" although
// the framework could hand out gigabytes.  The same holds for a process running under a fixed memory
// budget (an MPS client with a pinned-memory limit, a batch slot whose quota is spent), and for a
// latency-critical event loop that cannot afford the device-wide synchronisation cudaMalloc / cudaFree
// imply.  alphas_grid_load needs a few KB of device memory for the node table it derives (ln of the
// nodes, interval records); this entry point keeps that table in a fixed array inside the library's
// own image instead, so it calls no cudaMalloc, no cudaFree and no routine that allocates.
//
// The array below exists once on EVERY device that loads the library, from load until the process
// exits (PDFB_STATIC_SCRATCH_BYTES = 22 KB each).  All calls on one device share it, and it keeps
// what the last call left there.
//
// In HOST code the name `g_static_scratch` is only a handle for the runtime: it is not an address on
// the device, and handing it to a kernel (or to pdfb_setup_ln below) would make the kernel fault or
// read host memory.  The device address comes from cudaGetSymbolAddress, once per device with that
// device current (static_scratch_of); host code below only ever uses that pointer.
#include <cmath>
#include <cstring>
#include <mutex>

#include "pdfb_internal.cuh"

// layout of the scratch, for a node list of K <= PDFB_STATIC_MAX_KNOTS nodes (all offsets are
// fixed, computed for the maximum, so they do not depend on K):
//   [0)        q2k  K doubles   Q^2 of the nodes
//   [S)        a    K doubles   alpha_s at the nodes
//   [2S)       z    K doubles   ln Q^2 of the nodes (pdfb_ln, the function the queries use)
//   [3S)       rec  K records   IntervalRec of every interval (K1's rule, reading O2)
// with S = 8 * PDFB_STATIC_MAX_KNOTS bytes.
#define STATIC_S ((size_t)8 * PDFB_STATIC_MAX_KNOTS)
#define STATIC_BYTES (3 * STATIC_S + sizeof(IntervalRec) * PDFB_STATIC_MAX_KNOTS)
static_assert(STATIC_BYTES == PDFB_STATIC_SCRATCH_BYTES, "pdfb200.h states the size of the static scratch");

static __device__ __align__(256) unsigned char g_static_scratch[STATIC_BYTES];

// The node list travels as a kernel argument (4 KB; no copy call, nothing to stage, stream-ordered).
struct StaticNodes {
    double q2[PDFB_STATIC_MAX_KNOTS];
    double a[PDFB_STATIC_MAX_KNOTS];
};

// Writes the caller's nodes into the scratch.  `scratch` is the pointer cudaGetSymbolAddress gave.
__global__ void k_alphas_static_nodes(const __grid_constant__ StaticNodes nodes, int K, unsigned char *scratch)
{
    double *q2k = reinterpret_cast<double *>(scratch);
    double *a = reinterpret_cast<double *>(scratch + STATIC_S);
    for (int k = threadIdx.x; k < K; k += blockDim.x) { q2k[k] = nodes.q2[k]; a[k] = nodes.a[k]; }
}

// k_alphas (alphas_kernels.cu) with its node table in the static scratch: A.q2k / A.a / A.rec point
// into g_static_scratch.  Same search, same weights4, same ln, same contraction order, so the result
// is the one alphas_q2 gives through k_alphas, bit for bit (reading O6).
__global__ void __launch_bounds__(256)
k_alphas_static(const __grid_constant__ AlphasDev A, long long n, const double *__restrict__ q2, double *__restrict__ out)
{
    __shared__ __align__(16) IntervalRec rec[PDFB_STATIC_MAX_KNOTS];
    __shared__ double q2k[PDFB_STATIC_MAX_KNOTS], al[PDFB_STATIC_MAX_KNOTS];
    for (int e = threadIdx.x; e < A.K * 8; e += blockDim.x)
        reinterpret_cast<double *>(rec)[e] = reinterpret_cast<const double *>(A.rec)[e];
    for (int e = threadIdx.x; e < A.K; e += blockDim.x) { q2k[e] = A.q2k[e]; al[e] = A.a[e]; }
    __syncthreads();

    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < n; p += stride) {
        const double qv = __ldcs(q2 + p);
        double res;
        if (!(qv > 0.0)) {
            res = __longlong_as_double(0x7ff8000000000000LL);
        } else if (qv < A.q2_min) {
            res = A.a_first;
        } else if (qv > A.q2_max) {
            res = A.a_last;
        } else {
            int s = 0;
            for (int r = 1; r < A.n_sub; r++) if (A.q2_lo[r] <= qv) s = r;
            int lo = A.off[s];
            const int hi = A.off[s + 1] - 1;
            int top = hi - 1;
            while (top - lo > 0) {  // largest m in [lo, top] with q2k[m] <= qv
                const int mid = (lo + top + 1) >> 1;
                if (q2k[mid] <= qv) lo = mid; else top = mid - 1;
            }
            const IntervalRec r = rec[lo];
            double w[4];
            weights4(r, (pdfb_ln(qv) - r.z0) * r.inv_dz, w);
            const int i0 = max(lo - 1, A.off[s]), i3 = min(lo + 2, hi);  // absent knots: weight exactly 0
            res = fma(w[3], al[i3], fma(w[2], al[lo + 1], fma(w[1], al[lo], w[0] * al[i0])));
        }
        __stcs(out + p, res);
    }
}

// Device address of g_static_scratch on the CURRENT device, and that device's SM count.  Looked up
// on the first call per device (with that device current, as cudaGetSymbolAddress resolves the symbol
// for the current device) and remembered.
static int static_scratch_of(unsigned char **scratch, int *sms)
{
    static std::mutex mu;
    static unsigned char *ptr_of[64];
    static int sms_of[64];
    int dev = -1;
    PDFB_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return PDFB_ECUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr_of[dev]) {
        unsigned char *p = nullptr;
        int n_sm = 0;
        PDFB_CUDA(cudaGetSymbolAddress((void **)&p, g_static_scratch));
        PDFB_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        if (!p || n_sm < 1) return PDFB_ECUDA;
        sms_of[dev] = n_sm;
        ptr_of[dev] = p;
    }
    *scratch = ptr_of[dev];
    *sms = sms_of[dev];
    return PDFB_OK;
}

extern "C" int alphas_q2_static(int n_knots, const double *q_knots, const double *alphas, long long n,
                                const double *q2, double *out, void *cuda_stream)
{
    if (!q_knots || !alphas || n_knots < 2 || n < 0) return PDFB_EINVAL;
    if (n > 0 && (!q2 || !out)) return PDFB_EINVAL;
    if (n_knots > PDFB_STATIC_MAX_KNOTS) return PDFB_ESTATIC;  // the node table would not fit the static scratch
    // the node list is checked exactly as alphas_grid_load checks it (host arrays, nothing on the heap)
    StaticNodes nodes;
    AlphasDev d;
    memset(&d, 0, sizeof(d));
    int n_sub = 0;
    d.off[0] = 0;
    for (int k = 0; k < n_knots; k++) {
        if (!(q_knots[k] > 0.0) || !std::isfinite(q_knots[k]) || !std::isfinite(alphas[k])) return PDFB_EKNOTS;
        if (k && q_knots[k] < q_knots[k - 1]) return PDFB_EKNOTS;
        if (k && q_knots[k] == q_knots[k - 1]) {  // a repeated node: a flavour threshold, a new sub-grid
            if (++n_sub >= PDFB_MAX_SUBGRIDS) return PDFB_ELIMIT;
            d.off[n_sub] = k;
        }
        nodes.q2[k] = q_knots[k] * q_knots[k];
        nodes.a[k] = alphas[k];
    }
    d.off[++n_sub] = n_knots;
    for (int s = 0; s < n_sub; s++) if (d.off[s + 1] - d.off[s] < 2) return PDFB_EKNOTS;
    if (!(nodes.q2[0] >= 1e-300)) return PDFB_EKNOTS;  // subnormal scale
    for (int k = n_knots; k < PDFB_STATIC_MAX_KNOTS; k++) nodes.q2[k] = nodes.a[k] = 0.0;
    if (n == 0) return PDFB_OK;

    unsigned char *scratch = nullptr;  // device address of g_static_scratch (NOT the symbol itself)
    int sms = 0;
    int rc = static_scratch_of(&scratch, &sms);
    if (rc) return rc;
    double *d_q2k = reinterpret_cast<double *>(scratch);
    double *d_a = reinterpret_cast<double *>(scratch + STATIC_S);
    double *d_z = reinterpret_cast<double *>(scratch + 2 * STATIC_S);
    IntervalRec *d_rec = reinterpret_cast<IntervalRec *>(scratch + 3 * STATIC_S);

    d.K = n_knots; d.n_sub = n_sub;
    for (int s = 0; s < n_sub; s++) d.q2_lo[s] = nodes.q2[d.off[s]];
    d.q2_min = nodes.q2[0]; d.q2_max = nodes.q2[n_knots - 1];
    d.a_first = alphas[0]; d.a_last = alphas[n_knots - 1];
    d.q2k = d_q2k; d.a = d_a; d.rec = d_rec;

    // Every byte the evaluation reads (K nodes, K logarithms, K records: k1_interval_records writes the
    // pad record of each sub-grid too) is rewritten here, in stream order, before it is read: nothing in
    // the scratch has to start at zero, and what an earlier call left beyond entry K is never touched.
    cudaStream_t st = (cudaStream_t)cuda_stream;
    k_alphas_static_nodes<<<1, 256, 0, st>>>(nodes, n_knots, scratch);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    rc = pdfb_setup_ln(d_q2k, d_z, n_knots, st);
    if (!rc) rc = pdfb_setup_records(d_z, d_rec, nullptr, n_sub, d.off, st);
    if (rc) return rc;
    long long blocks = (n + 255) / 256;
    if (blocks > (long long)sms * 8) blocks = (long long)sms * 8;
    k_alphas_static<<<(unsigned)blocks, 256, 0, st>>>(d, n, q2, out);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
