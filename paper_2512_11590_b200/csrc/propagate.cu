// propagate.cu -- R-matrix propagation over sub-intervals (PAPER.md:53 "propagation", :327 hprmat_init(nr, ns, rmax, zrma)
// with ns sub-intervals; the paper defers the formulas to its ref. [2]; reading R16 in DESIGN.md section 3).
//
// On the sub-interval (a_lo, a_hi) the Bloch operator acts at BOTH ends, and the solution values at the two ends follow from
// the outward derivatives through the four Nc x Nc "sector" matrices
//     Rsec_ab = (hbar^2/2mu) B_a^T (C - E I)^-1 B_b,   a, b in {L, R},   B_a[(c,i),c'] = f_i(a_a) delta_cc'
// (hprmat_solve_sector):   u(a_hi) = Rsec_RR u'(a_hi) - Rsec_RL u'(a_lo),   u(a_lo) = Rsec_LR u'(a_hi) - Rsec_LL u'(a_lo).
// With the R-matrix at a_lo, u(a_lo) = a_lo R_in u'(a_lo), eliminating u'(a_lo) gives the R-matrix at a_hi:
//     a_hi R_out = Rsec_RR - Rsec_RL (Rsec_LL + a_lo R_in)^-1 Rsec_LR.
// This file does that Nc x Nc algebra on the device with the library's own FP64 LU (lu.cu) and DMMA GEMM (zgemm.cu).
#include <atomic>
#include <cstdio>

#include "lu.cuh"

namespace hp {

int zgemm(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, const double2 *B, long ldb,
          double beta, double2 *C, long ldc);

namespace {

inline size_t up256(size_t b) { return (b + 255) / 256 * 256; }

// M <- Rsec_LL + a_lo R_in;  Y <- Rsec_LR;  Rout <- Rsec_RR / a_hi
__global__ void __launch_bounds__(256) propagate_prepare_kernel(long nn, double a_lo, double a_hi, const double2 *__restrict__ Rin,
                                                                const double2 *__restrict__ Rsec, double2 *__restrict__ M,
                                                                double2 *__restrict__ Y, double2 *__restrict__ Rout) {
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < nn; i += (long)gridDim.x * blockDim.x) {
        const double2 ll = Rsec[i], lr = Rsec[nn + i], rr = Rsec[3 * nn + i], r = Rin[i];
        M[i] = make_double2(ll.x + a_lo * r.x, ll.y + a_lo * r.y);
        Y[i] = lr;
        Rout[i] = make_double2(rr.x / a_hi, rr.y / a_hi);
    }
}

}  // namespace
}  // namespace hp

using namespace hp;

extern "C" size_t hprmat_propagate_workspace_bytes(int nch) {
    if (nch < 0) return 0;
    const size_t n = (size_t)nch;
    return 2 * up256(n * n * sizeof(double2)) + up256(n * sizeof(int)) + 256 + LuWork<ZView>::bytes(nch);
}

extern "C" int hprmat_propagate(void *cuda_stream, int nch, double a_lo, double a_hi, const void *R_in, const void *Rsec,
                                void *R_out, int *info_dev, void *workspace, size_t workspace_bytes) {
    if (nch < 1) return -2;
    if (!(a_lo > 0.0)) return -3;
    if (!(a_hi > a_lo)) return -4;
    if (!R_in) return -5;
    if (!Rsec) return -6;
    if (!R_out) return -7;
    if (!info_dev) return -8;
    if (!workspace || ((uintptr_t)workspace & 255)) return -9;
    if (workspace_bytes < hprmat_propagate_workspace_bytes(nch)) return HPRMAT_ENOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long nn = (long)nch * nch;
    char *p = (char *)workspace;
    double2 *M = (double2 *)p;  p += up256((size_t)nn * sizeof(double2));
    double2 *Y = (double2 *)p;  p += up256((size_t)nn * sizeof(double2));
    int *ipiv = (int *)p;       p += up256((size_t)nch * sizeof(int)) + 256;
    LuWork<ZView> wk;
    wk.carve(p, nch);
    HP_CUDA(cudaMemsetAsync(info_dev, 0, sizeof(int), st));
    propagate_prepare_kernel<<<(int)std::min<long>((nn + 255) / 256, 148 * 8), 256, 0, st>>>(
        nn, a_lo, a_hi, (const double2 *)R_in, (const double2 *)Rsec, M, Y, (double2 *)R_out);
    HP_LAUNCHED();
    HP_TRY(getrf<ZView>(st, nch, ZView(M, nch), ipiv, info_dev, wk));
    HP_TRY(getrs<ZView>(st, nch, nch, ZView(M, nch), ZView(Y, nch), wk));
    // R_out <- R_out - (1/a_hi) Rsec_RL Y
    return zgemm(st, nch, nch, nch, -1.0 / a_hi, (const double2 *)Rsec + 2 * nn, nch, Y, nch, 1.0, (double2 *)R_out, nch);
}

// ---- the same propagation step for callers that may not allocate (code under CUDA-graph capture, serving loops, harnesses
// that forbid cudaMalloc): the workspace of hprmat_propagate lives in a file-scope device array instead of a caller's buffer.
// Every GPU that loads the library holds PROP_STATIC_BYTES (3 MiB) until the process exits.  ONE array per device, shared by
// every call and keeping the last call's contents: calls whose GPU work may overlap (different streams, several host
// threads) race on it -- serialise them, or use hprmat_propagate with a workspace per call.
namespace hp {
namespace {
constexpr int PROP_STATIC_MAX_NCH = 128;  // = LEAF: the nch x nch LU then keeps no solve-block inverses and forks no side stream
constexpr size_t PROP_STATIC_BYTES = 3u << 20;
static __device__ __align__(256) unsigned char g_prop_scratch[PROP_STATIC_BYTES];

// In host code g_prop_scratch is a host-side stand-in, not a device address: the address a kernel may use comes from
// cudaGetSymbolAddress, asked once per device with that device current.
std::atomic<void *> g_prop_scratch_addr[32];
int prop_scratch(void **out) {
    int dev = 0;
    HP_CUDA(cudaGetDevice(&dev));
    const bool tracked = dev >= 0 && dev < 32;
    void *p = tracked ? g_prop_scratch_addr[dev].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        HP_CUDA(cudaGetSymbolAddress(&p, g_prop_scratch));
        if (tracked) g_prop_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return 0;
}
}  // namespace
}  // namespace hp

extern "C" int hprmat_propagate_static_max_nch(void) { return PROP_STATIC_MAX_NCH; }

extern "C" int hprmat_propagate_static(void *cuda_stream, int nch, double a_lo, double a_hi, const void *R_in, const void *Rsec,
                                       void *R_out, int *info_dev) {
    if (nch < 1) return -2;
    if (nch > PROP_STATIC_MAX_NCH || hprmat_propagate_workspace_bytes(nch) > PROP_STATIC_BYTES) {
        snprintf(g_cuda_err, sizeof(g_cuda_err),
                 "hprmat_propagate_static: nch = %d exceeds the static scratch limit nch <= %d (use hprmat_propagate with a workspace)",
                 nch, PROP_STATIC_MAX_NCH);
        return HPRMAT_ENOMEM;
    }
    void *scratch = nullptr;
    HP_TRY(prop_scratch(&scratch));
    // The array keeps the previous call's contents (possibly of another nch).  The LU clears its own counters, lock words and
    // verdict word on every call (lu.cu getrf) and M, Y and the pivot table are written before they are read; the whole array
    // is cleared here all the same (3 MiB, ~2 us on the caller's stream) so that a call's result cannot depend on its
    // predecessor's leftovers.
    HP_CUDA(cudaMemsetAsync(scratch, 0, PROP_STATIC_BYTES, (cudaStream_t)cuda_stream));
    return hprmat_propagate(cuda_stream, nch, a_lo, a_hi, R_in, Rsec, R_out, info_dev, scratch, PROP_STATIC_BYTES);
}
