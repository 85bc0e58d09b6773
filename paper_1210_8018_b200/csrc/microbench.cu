// microbench.cu -- measured FP64 FMA rate of the device, the denominator of the "alu" roofline that
// bench.py reports for the one kernel of the path that is bound by plain FP64 arithmetic (the ACCUM_G
// measure kernel; flop counts of Table 1, are why it matters).
// Not on the gauge-fixing path: a debug entry point of the C ABI (lgf_debug_dfma_rate).
#include <cuda_runtime.h>

#include "../../include/lgf.h"

namespace {

// CHAINS independent dependent-FMA chains per thread: enough instruction-level parallelism to keep the
// FP64 pipe issuing every cycle it can, no memory traffic inside the loop.
template <int CHAINS>
__global__ void __launch_bounds__(256) k_dfma(double *out, int iters, double a, double b)
{
    double x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; c++) x[c] = (double)(threadIdx.x + c) * 1e-3;
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int u = 0; u < 8; u++)
#pragma unroll
            for (int c = 0; c < CHAINS; c++) x[c] = fma(x[c], a, b);
    }
    double s = 0;
#pragma unroll
    for (int c = 0; c < CHAINS; c++) s += x[c];
    if (s == 123.456) out[0] = s;      // never true: keeps the chains alive
}

} // namespace

extern "C" int lgf_debug_dfma_rate(void *cuda_stream, double *dfma_per_second)
{
    if (!dfma_per_second) return LGF_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LGF_ERR_CUDA;
    double *d = nullptr;
    if (cudaMalloc(&d, sizeof(double)) != cudaSuccess) return LGF_ERR_CUDA;   // debug call only: never on the hot path
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    constexpr int CHAINS = 8;
    const int blocks = sms * 8, iters = 4096;
    double best = 0;
    for (int rep = 0; rep < 5; rep++) {
        cudaEventRecord(e0, st);
        k_dfma<CHAINS><<<blocks, 256, 0, st>>>(d, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double n = (double)blocks * 256.0 * (double)iters * 8.0 * CHAINS;
        if (rep > 0 && ms > 0 && n / (ms * 1e-3) > best) best = n / (ms * 1e-3);   // first launch is the warm-up
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d);
    if (cudaGetLastError() != cudaSuccess || best <= 0) return LGF_ERR_CUDA;
    *dfma_per_second = best;
    return LGF_OK;
}
