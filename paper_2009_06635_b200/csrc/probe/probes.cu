// probes.cu -- two machine probes behind a C-ABI of their own (libpdfb200_probe.so: pdfb_probe), used by bench.py to put MEASURED
// denominators under the two bounds that MEASURED_PEAKS.json does not carry ("the
// build must measure" the FP64 peak):
//   PDFB_PROBE_FP64  independent DFMA chains at full occupancy -> FP64-pipe warp instructions x 32 / s
//   PDFB_PROBE_LDS   conflict-free LDS.128 in the gather's own rotated pattern -> shared-memory bytes / s
// They evaluate nothing of the method and are not on the product path.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../../include/pdfb200_probe.h"

#define PROBE_OK 0
#define PROBE_EINVAL (-1)
#define PROBE_ECUDA (-4)
#define PROBE_CUDA(call) do { if ((call) != cudaSuccess) return PROBE_ECUDA; } while (0)

__global__ void __launch_bounds__(512, 2) k_probe_dfma(double *out, int iters)
{
    double a[8];
#pragma unroll
    for (int k = 0; k < 8; k++) a[k] = 1.0 + 1e-9 * (threadIdx.x + k);
    const double m = 1.0 - 1e-12, c = 1e-13;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int k = 0; k < 8; k++) a[k] = fma(a[k], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 8; k++) s += a[k];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(512, 1) k_probe_lds(double *out, int iters, int smem_bytes)
{
    extern __shared__ __align__(128) unsigned char sm[];
    for (int i = threadIdx.x; i < smem_bytes / 8; i += blockDim.x) reinterpret_cast<double *>(sm)[i] = 1.0;
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(sm);
    const uint32_t nlines = (uint32_t)smem_bytes / 128u;
    uint32_t rng = threadIdx.x * 2654435761u + blockIdx.x * 40503u + 12345u;
    const int lane8 = threadIdx.x & 7;
    double acc = 0.0;
    for (int it = 0; it < iters; it++) {
        rng = rng * 1664525u + 1013904223u;
        const uint32_t a0 = base + ((rng >> 8) % nlines) * 128u;  // a random 128-byte line per lane
#pragma unroll
        for (int s = 0; s < 8; s++) {  // its 8 chunks, each quarter-warp on 8 distinct bank groups
            double x, y;
            asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a0 + (uint32_t)(((s + lane8) & 7) << 4)));
            acc += x;
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

extern "C" int pdfb_probe(int which, int device, double *result)
{
    if (!result) return PROBE_EINVAL;
    *result = 0.0;
    int ndev = 0, sms = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return PROBE_ECUDA;
    PROBE_CUDA(cudaSetDevice(device));
    PROBE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    double *buf = nullptr;
    PROBE_CUDA(cudaMalloc(&buf, sizeof(double) * (size_t)sms * 2 * 512));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int rc = PROBE_OK;
    float best = 1e30f;
    double work = 0.0;
    if (which == PDFB_PROBE_FP64) {
        const int iters = 40000;
        for (int rep = 0; rep < 4; rep++) {  // first repetition warms up
            cudaEventRecord(e0); k_probe_dfma<<<sms * 2, 512>>>(buf, iters); cudaEventRecord(e1);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = PROBE_ECUDA; break; }
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            if (rep && ms < best) best = ms;
        }
        work = (double)sms * 2 * 512 * 8.0 * iters;  // thread-level DFMA = FP64 lane operations
    } else if (which == PDFB_PROBE_LDS) {
        const int iters = 20000, smem = 200 * 1024;
        if (cudaFuncSetAttribute(k_probe_lds, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) rc = PROBE_ECUDA;
        for (int rep = 0; rep < 4 && !rc; rep++) {
            cudaEventRecord(e0); k_probe_lds<<<sms, 512, smem>>>(buf, iters, smem); cudaEventRecord(e1);
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = PROBE_ECUDA; break; }
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            if (rep && ms < best) best = ms;
        }
        work = (double)sms * 512 * 8.0 * 16.0 * iters;  // bytes delivered to registers
    } else {
        rc = PROBE_EINVAL;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(buf);
    if (cudaGetLastError() != cudaSuccess) rc = rc ? rc : PROBE_ECUDA;
    if (!rc) *result = work / (best * 1e-3);
    return rc;
}
