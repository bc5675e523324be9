// dmma_peak.cu -- bench.py's measurement of the FP64 tensor-core (DMMA) issue-rate ceiling of this GPU, the denominator of
// the FP64 trailing-update roofline.  Built into libhprmat_bench.so, which only bench.py loads; the
// product library does not contain it.  A register-resident loop of independent mma.sync.m8n8k4.f64 chains, no memory
// traffic: every SM sub-partition is kept saturated by 8 warps x 8 independent accumulators.
#include <cuda_runtime.h>

#include "../../include/hprmat_profile.h"

namespace {

__global__ void __launch_bounds__(256) dmma_peak_kernel(int iters, double *sink) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = 0.0;
    double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 12345.678) sink[0] = s;  // keeps the chain alive; never true in practice
}

}  // namespace

// Runs the loop on ctas_per_sm x 148 CTAs of 8 warps; *tflops = real flops (2*8*8*4 per MMA) / device time.
extern "C" int hprmat_bench_dmma_peak(void *cuda_stream, int iters, int ctas_per_sm, double *tflops, double *ms_out) {
    if (iters < 1) return -2;
    if (ctas_per_sm < 1) return -3;
    if (!tflops) return -4;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaMalloc((void **)&sink, sizeof(double)) != cudaSuccess || cudaEventCreate(&e0) != cudaSuccess ||
        cudaEventCreate(&e1) != cudaSuccess)
        return 4;
    const int grid = 148 * ctas_per_sm;
    dmma_peak_kernel<<<grid, 256, 0, st>>>(iters / 8 + 1, sink);  // warm-up
    cudaEventRecord(e0, st);
    dmma_peak_kernel<<<grid, 256, 0, st>>>(iters, sink);
    cudaEventRecord(e1, st);
    const cudaError_t rc = cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = (double)grid * 8 /*warps*/ * (double)iters * 8 /*mma per iter*/ * 512.0;
    *tflops = ms > 0.f ? flops / (ms * 1e-3) * 1e-12 : 0.0;
    if (ms_out) *ms_out = ms;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return rc == cudaSuccess ? 0 : 4;
}
