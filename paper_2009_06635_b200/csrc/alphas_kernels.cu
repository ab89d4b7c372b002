// alphas_kernels.cu -- K4: alpha_s(Q^2) by cubic Hermite interpolation in ln Q^2 with constant
// extrapolation (reading O6; "log-cubic interpolation with constant extrapolation
// from the (alpha_s(Q), Q) nodes ... improved treatment of the sub-grids mechanism").
// The whole node table (knots, values, interval records: 80 B per node) lives in shared memory.
#include "pdfb_internal.cuh"

#define ALPHAS_SMEM_MAX_KNOTS 512

__global__ void __launch_bounds__(256)
k_alphas(AlphasDev A, long long n, const double *__restrict__ q2, double *__restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    IntervalRec *rec = reinterpret_cast<IntervalRec *>(smem_raw);
    double *q2k = reinterpret_cast<double *>(rec + A.K);
    double *al = q2k + A.K;
    for (int e = threadIdx.x; e < A.K * 8; e += blockDim.x)
        reinterpret_cast<double *>(rec)[e] = reinterpret_cast<const double *>(A.rec)[e];
    for (int e = threadIdx.x; e < A.K; e += blockDim.x) { q2k[e] = A.q2k[e]; al[e] = A.a[e]; }
    __syncthreads();

    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < n; p += stride) {
        double qv = __ldcs(q2 + p);
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
            int lo = A.off[s], hi = A.off[s + 1] - 1;  // cell index in [lo, hi-1]
            int top = hi - 1;
            while (top - lo > 0) {                     // largest m in [lo, top] with q2k[m] <= qv
                int mid = (lo + top + 1) >> 1;
                if (q2k[mid] <= qv) lo = mid; else top = mid - 1;
            }
            const IntervalRec r = rec[lo];
            double w[4];
            weights4(r, (pdfb_ln(qv) - r.z0) * r.inv_dz, w);
            // knots lo-1 .. lo+2; absent ones have weight exactly 0, clamp their index
            int i0 = max(lo - 1, A.off[s]), i3 = min(lo + 2, hi);
            res = fma(w[3], al[i3], fma(w[2], al[lo + 1], fma(w[1], al[lo], w[0] * al[i0])));
        }
        __stcs(out + p, res);
    }
}

int pdfb_launch_alphas(const pdfb_alphas *a, long long n, const double *q2, double *out, cudaStream_t st)
{
    if (n == 0) return PDFB_OK;
    size_t smem = (size_t)a->d.K * (sizeof(IntervalRec) + 16);
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    k_alphas<<<(unsigned)blocks, 256, smem, st>>>(a->d, n, q2, out);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
