// xfxq2_kernels.cu -- K2/K3: knot location + evaluation of xf(x,Q^2) (readings O3-O5).
//
// v0 (reference CUDA path): one thread per query point, tables through the read-only cache.
// Per point: classify, sub-grid select, binary search on raw x / Q^2 knots, two logs, the
// eight 1-D weights; then per requested flavour a 16-term contraction of the 4x4 value
// stencil ("log-bicubic PDF interpolation in terms of x and Q^2").
#include "xfxq2_v0.cuh"

__global__ void __launch_bounds__(256)
k_xfxq2_v0(GridDev g, ReqCols rc, long long n, const double *__restrict__ x, const double *__restrict__ q2,
           double *__restrict__ out, long long out_stride, int mode, int member0)
{
    long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (p >= n) return;
    // blockIdx.y = member of the set: its table, and its block of rc.n output rows
    const double *val = g.val + (long long)(member0 + blockIdx.y) * g.val_mstride;
    const long long mo = (long long)blockIdx.y * rc.n * out_stride;  // elements (doubles, or floats for fp32 output)
    double xv = x[p], qv = q2[p];
    if (mode & 1) qv = (qv > 0.0) ? qv * qv : -1.0;  // Q in GeV -> Q^2 (a non-positive Q is invalid)
    double res[PDFB_MAX_PIDS];
    const bool ok = xf_point_v0(g, val, rc, xv, qv, res);
    const int om = mode >> 1;  // output layout, as the shared-memory kernel's OUT (xfxq2_smem.cuh)
    for (int r = 0; r < rc.n; r++) {
        if (om == 0) out[mo + r * out_stride + p] = res[r];
        else if (om == 1) out[mo + p * rc.n + r] = res[r];
        else reinterpret_cast<float *>(out)[mo + r * out_stride + p] = (float)res[r];
    }
    if (!ok && blockIdx.y == 0) atomicAdd(g.n_invalid, 1ULL);
}

int pdfb_launch_xfxq2(const pdfb_grid *g, int n_req, const int *cols, long long n, const double *x,
                      const double *q2, double *out, long long out_stride, cudaStream_t st, int mode, int member0, int n_mem)
{
    if (n == 0 || n_mem == 0) return PDFB_OK;
    if (g->d.smem_ok) return pdfb_launch_xfxq2_smem(g, n_req, cols, n, x, q2, out, out_stride, st, mode, member0, n_mem);
    ReqCols rc;
    rc.n = n_req;
    for (int r = 0; r < n_req; r++) rc.col[r] = cols[r];
    long long blocks = (n + 255) / 256;
    if (n_mem > 65535) return PDFB_ELIMIT;
    k_xfxq2_v0<<<dim3((unsigned)blocks, (unsigned)n_mem), 256, 0, st>>>(g->d, rc, n, x, q2, out, out_stride, mode, member0);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
