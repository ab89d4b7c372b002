// alphas_kernels.cu -- K4: alpha_s(Q^2) by cubic Hermite interpolation in ln Q^2 with constant
// extrapolation (reading O6; "log-cubic interpolation with constant extrapolation
// from the (alpha_s(Q), Q) nodes ... improved treatment of the sub-grids mechanism").
// The whole node table (knots, values, interval records: 80 B per node) lives in shared memory.
#include <atomic>

#include "pdfb_internal.cuh"

#define ALPHAS_SMEM_MAX_KNOTS 512

__global__ void __launch_bounds__(256)
k_alphas(AlphasDev A, long long n, const double *__restrict__ q2, double *__restrict__ out, int q_is_q)
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
        if (q_is_q) qv = (qv > 0.0) ? qv * qv : -1.0;
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

// Fast path (K <= 192 nodes): replicated coefficient lines in shared memory, LUT location,
// one cubic in s = ln Q^2 - Z_m per point (five doubles per interval: two LDS.128 and one LDS.64),
// ln Q^2 through a 64-entry table (ln_tab, pdfb_internal.cuh).  Six points per thread and iteration;
// 2 CTAs of 768 threads per SM (48 KB of tables each).  Measured per 1e8 points (threads x CTAs x
// points): 512 x 3 x 4: 0.328 ms, 512 x 3 x 8: 0.324, 768 x 2 x 4: 0.320, 768 x 2 x 6: 0.312 (kept),
// 768 x 2 x 8: 0.312, 640 x 2 x 6: 0.324, 1024 x 1 x 8: 0.333, 384 x 4 x 4: 0.332, 256 x 6 x 4: 0.436.
#ifndef NT_ALPHAS
#define NT_ALPHAS 768
#endif
#ifndef CTAS_ALPHAS
#define CTAS_ALPHAS 2
#endif
#ifndef PTS_ALPHAS
#define PTS_ALPHAS 6   // points per thread and iteration
#endif

template <bool Q_IS_Q>
__global__ void __launch_bounds__(NT_ALPHAS, CTAS_ALPHAS)
k_alphas_fast(const __grid_constant__ AlphasDev A, long long n, const double *__restrict__ q2,
              double *__restrict__ out)
{
    extern __shared__ __align__(128) unsigned char smem[];
    for (int e = threadIdx.x; e < A.fast_bytes / 16; e += NT_ALPHAS)
        reinterpret_cast<int4 *>(smem)[e] = __ldg(reinterpret_cast<const int4 *>(A.fast) + e);
    __syncthreads();
    const uint32_t lines = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)((threadIdx.x & 7) << 4);
    const uint32_t lntab = lines + (uint32_t)A.f_lntab;
    const uint32_t d3_off = 256u + ((uint32_t)(threadIdx.x & 15) << 3) - ((uint32_t)(threadIdx.x & 7) << 4);  // line 2, copy lane & 15
    const double *q2k = reinterpret_cast<const double *>(smem + A.f_q2k);
    const unsigned short *lut = reinterpret_cast<const unsigned short *>(smem + A.f_lut);
    const double qnan = __longlong_as_double(0x7ff8000000000000LL);
    auto eval = [&](double qv) -> double {
        double res;
        if (Q_IS_Q) qv = (qv > 0.0) ? qv * qv : -1.0;  // Q in GeV -> Q^2
        if (qv >= A.q2_min && qv < A.q2_max) {  // (Q^2 = the last node takes the frozen branch: the node value, bit for bit)
            double2 le;  // {1/c, ln c} of qv's mantissa bin
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(le.x), "=d"(le.y) : "r"(lntab + (uint32_t)ln_tab_bin(qv) * 128u));
            const double v = ln_tab(qv, le);
            int b = min(max((int)((v - A.lut_v0) * A.lut_inv_h), 0), PDFB_LUT_BINS - 1);
            const int e = lut[b], d = (e >> 1) & 3;
            int m = e >> 3;
            if (d) { if (q2k[m + d] <= qv) m += d; }
            if (e & 1)
                while (m < A.K - 1 && q2k[m + 1] <= qv) ++m;
            m = min(m, A.K - 2);
            const uint32_t rec = lines + (uint32_t)m * (uint32_t)PDFB_ALPHAS_LINE;
            double2 zd, d12;
            double d3;
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(zd.x), "=d"(zd.y) : "r"(rec));
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(d12.x), "=d"(d12.y) : "r"(rec + 128u));
            asm volatile("ld.shared.f64 %0, [%1];" : "=d"(d3) : "r"(rec + d3_off));
            const double s = v - zd.x;
            res = fma(s, fma(s, fma(s, d3, d12.y), d12.x), zd.y);
        } else {
            res = (qv < A.q2_min) ? A.a_first : A.a_last;
        }
        return (qv > 0.0) ? res : qnan;  // NaN and non-positive Q^2 have no value
    };
    // PTS_ALPHAS points per thread and iteration: the loads go out together, the ln chains interleave.
    // (Measured and dropped: the four points evaluated stage by stage without branches between the
    // stages -- all table loads of a stage issued together -- 0.345 ms against 0.330 ms per 1e8 points.)
    const long long stride = (long long)gridDim.x * NT_ALPHAS;
    long long p = blockIdx.x * (long long)NT_ALPHAS + threadIdx.x;
    for (; p + (PTS_ALPHAS - 1) * stride < n; p += PTS_ALPHAS * stride) {
        double q[PTS_ALPHAS], r[PTS_ALPHAS];
#pragma unroll
        for (int k = 0; k < PTS_ALPHAS; k++) q[k] = __ldcs(q2 + p + k * stride);
#pragma unroll
        for (int k = 0; k < PTS_ALPHAS; k++) r[k] = eval(q[k]);
#pragma unroll
        for (int k = 0; k < PTS_ALPHAS; k++) __stcs(out + p + k * stride, r[k]);
    }
    for (; p < n; p += stride) __stcs(out + p, eval(__ldcs(q2 + p)));
}

int pdfb_launch_alphas(const pdfb_alphas *a, long long n, const double *q2, double *out, cudaStream_t st, int q_is_q)
{
    if (n == 0) return PDFB_OK;
    if (a->d.fast_ok) {
        // the attribute is per function and device; setting it twice is harmless, so a relaxed
        // per-device bit is enough for concurrent callers
        static std::atomic<unsigned long long> attr_done{0};
        const unsigned long long bit = 1ULL << (a->device & 63);
        if (!(attr_done.load(std::memory_order_acquire) & bit)) {
            PDFB_CUDA(cudaFuncSetAttribute(k_alphas_fast<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024));
            PDFB_CUDA(cudaFuncSetAttribute(k_alphas_fast<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 110 * 1024));
            attr_done.fetch_or(bit, std::memory_order_release);
        }
        long long blocks = (n + NT_ALPHAS - 1) / NT_ALPHAS;
        if (blocks > (long long)a->sms * CTAS_ALPHAS) blocks = (long long)a->sms * CTAS_ALPHAS;
        if (q_is_q) k_alphas_fast<true><<<(unsigned)blocks, NT_ALPHAS, a->d.fast_bytes, st>>>(a->d, n, q2, out);
        else k_alphas_fast<false><<<(unsigned)blocks, NT_ALPHAS, a->d.fast_bytes, st>>>(a->d, n, q2, out);
        pdfb_count_launch(1);
        PDFB_CUDA(cudaGetLastError());
        return PDFB_OK;
    }
    size_t smem = (size_t)a->d.K * (sizeof(IntervalRec) + 16);
    long long blocks = (n + 255) / 256;
    if (blocks > (long long)a->sms * 8) blocks = (long long)a->sms * 8;
    k_alphas<<<(unsigned)blocks, 256, smem, st>>>(a->d, n, q2, out, q_is_q);
    pdfb_count_launch(1);
    PDFB_CUDA(cudaGetLastError());
    return PDFB_OK;
}
