// probe.cu -- measurement aid: the FP64 tensor-core (DMMA) issue-rate ceiling of this GPU, the denominator of the FP64
// trailing-update roofline.  A register-resident loop of independent mma.sync.m8n8k4.f64 chains,
// no memory traffic: every SM sub-partition is kept saturated by 8 warps x 8 independent accumulators.
#include "common.cuh"

namespace hp {

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

}  // namespace hp

// Runs the loop on ctas_per_sm x 148 CTAs of 8 warps; *tflops = real flops (2*8*8*4 per MMA) / device time.
extern "C" int hprmat_probe_dmma(void *cuda_stream, int iters, int ctas_per_sm, double *tflops, double *ms_out) {
    using namespace hp;
    if (iters < 1) return -2;
    if (ctas_per_sm < 1) return -3;
    if (!tflops) return -4;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double *sink = nullptr;
    HP_CUDA(cudaMalloc((void **)&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    HP_CUDA(cudaEventCreate(&e0));
    HP_CUDA(cudaEventCreate(&e1));
    const int grid = kNumSMs * ctas_per_sm;
    dmma_peak_kernel<<<grid, 256, 0, st>>>(iters / 8 + 1, sink);  // warm-up
    HP_LAUNCHED();
    HP_CUDA(cudaEventRecord(e0, st));
    dmma_peak_kernel<<<grid, 256, 0, st>>>(iters, sink);
    HP_LAUNCHED();
    HP_CUDA(cudaEventRecord(e1, st));
    HP_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = (double)grid * 8 /*warps*/ * (double)iters * 8 /*mma per iter*/ * 512.0;
    *tflops = flops / (ms * 1e-3) * 1e-12;
    if (ms_out) *ms_out = ms;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    return HPRMAT_OK;
}


namespace hp {
int probe_panel(cudaStream_t st, int m, int reps, float *A_re, float *A_im, long lda, void *work, double *us_per_panel,
                long long *phase_cycles_host);
}
// Panel-factorisation probe: see hprmat.h.
extern "C" int hprmat_probe_panel(void *cuda_stream, int m, int reps, float *A_re, float *A_im, int lda, void *workspace,
                                  double *us_per_panel, long long *phase_cycles) {
    if (m < 1) return -2;
    if (reps < 1) return -3;
    if (!A_re || !A_im) return -4;
    if (lda < m) return -6;
    if (!workspace) return -7;
    if (!us_per_panel) return -8;
    return hp::probe_panel((cudaStream_t)cuda_stream, m, reps, A_re, A_im, lda, workspace, us_per_panel, phase_cycles);
}
