// api_raw.cu -- raw dense complex entries of the C ABI: LU, triangular solves, workspace query (FP64 part).
// PAPER.md:119 ("all solvers take the matrix M and right-hand side b and return c"), :125-137 (ZGESV semantics).
#include <algorithm>

#include "lu.cuh"

using namespace hp;

namespace hp {
size_t raw_workspace_fp64(int n) { return LuWork<ZView>::bytes(n) + 256; }  // + one int for the zero-pivot flag
size_t raw_workspace_mixed(int n, int nrhs);
int zsolve_mixed(cudaStream_t st, int n, int nrhs, const double2 *A, long lda, double2 *B, long ldb, int *ipiv, bool refine,
                 int max_refine, double tol, void *workspace, hprmat_info *info);
}  // namespace hp

extern "C" size_t hprmat_workspace_bytes(int n, int nrhs, int mode) {
    if (n < 0 || nrhs < 0) return 0;
    if (mode == HPRMAT_MIXED || mode == HPRMAT_MIXED_REFINE) return std::max(raw_workspace_mixed(n, nrhs), raw_workspace_fp64(n));
    return raw_workspace_fp64(n);
}

extern "C" int hprmat_zgetrf(void *cuda_stream, int n, void *A, int lda, int *ipiv, int *info_dev, void *workspace,
                             size_t workspace_bytes) {
    if (n < 0) return -2;
    if (!A && n > 0) return -3;
    if (lda < (n > 1 ? n : 1)) return -4;
    if (!ipiv && n > 0) return -5;
    if (!info_dev) return -6;
    if (!workspace || ((uintptr_t)workspace & 255)) return -7;
    if (workspace_bytes < raw_workspace_fp64(n)) return HPRMAT_ENOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LuWork<ZView> wk;
    wk.carve(workspace, n);
    HP_CUDA(cudaMemsetAsync(info_dev, 0, sizeof(int), st));
    return getrf<ZView>(st, n, ZView((double2 *)A, lda), ipiv, info_dev, wk);
}

extern "C" int hprmat_zgetrs(void *cuda_stream, int n, int nrhs, const void *A, int lda, const int *ipiv, void *B,
                             int ldb, void *workspace, size_t workspace_bytes) {
    (void)ipiv;  // the interchanges are replayed from the per-batch net permutations kept in the workspace
    if (n < 0) return -2;
    if (nrhs < 0) return -3;
    if (!A && n > 0) return -4;
    if (lda < (n > 1 ? n : 1)) return -5;
    if (!B && n > 0 && nrhs > 0) return -7;
    if (ldb < (n > 1 ? n : 1)) return -8;
    if (!workspace || ((uintptr_t)workspace & 255)) return -9;
    if (workspace_bytes < raw_workspace_fp64(n)) return HPRMAT_ENOMEM;
    LuWork<ZView> wk;
    wk.carve(workspace, n);
    return getrs<ZView>((cudaStream_t)cuda_stream, n, nrhs, ZView((double2 *)A, lda), ZView((double2 *)B, ldb), wk);
}

extern "C" int hprmat_zsolve(void *cuda_stream, int n, int nrhs, void *A, int lda, void *B, int ldb, int *ipiv, int mode,
                             int max_refine, double tol, void *workspace, size_t workspace_bytes, hprmat_info *info) {
    if (n < 0) return -2;
    if (nrhs < 0) return -3;
    if (!A && n > 0) return -4;
    if (lda < (n > 1 ? n : 1)) return -5;
    if (!B && n > 0 && nrhs > 0) return -6;
    if (ldb < (n > 1 ? n : 1)) return -7;
    if (!ipiv && n > 0) return -8;
    if (mode != HPRMAT_FP64 && mode != HPRMAT_MIXED && mode != HPRMAT_MIXED_REFINE) return -9;
    if (!workspace || ((uintptr_t)workspace & 255)) return -12;
    if (workspace_bytes < hprmat_workspace_bytes(n, nrhs, mode)) return HPRMAT_ENOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (mode != HPRMAT_FP64) {
        if (info) {
            *info = hprmat_info();
            info->backward_err = -1.0;
        }
        if (n == 0 || nrhs == 0) return HPRMAT_OK;
        const int rc = zsolve_mixed(st, n, nrhs, (const double2 *)A, lda, (double2 *)B, ldb, ipiv, mode == HPRMAT_MIXED_REFINE,
                                    max_refine, tol, workspace, info);
        if (info) info->status = rc;
        return rc;
    }
    if (info) {
        *info = hprmat_info();
        info->backward_err = -1.0;  // A is overwritten by its factors in FP64 mode: no residual can be formed
    }
    if (n == 0) return HPRMAT_OK;
    LuWork<ZView> wk;
    const size_t used = wk.carve(workspace, n);
    int *info_dev = (int *)((char *)workspace + used);
    struct Events {  // destroyed on every return path
        cudaEvent_t e[3] = {nullptr, nullptr, nullptr};
        ~Events() {
            for (auto &x : e)
                if (x) cudaEventDestroy(x);
        }
    } evs;
    cudaEvent_t *ev = evs.e;
    if (info)
        for (auto &e : evs.e) HP_CUDA(cudaEventCreate(&e));
    HP_CUDA(cudaMemsetAsync(info_dev, 0, sizeof(int), st));
    if (info) HP_CUDA(cudaEventRecord(ev[0], st));
    HP_TRY(getrf<ZView>(st, n, ZView((double2 *)A, lda), ipiv, info_dev, wk));
    if (info) HP_CUDA(cudaEventRecord(ev[1], st));
    HP_TRY(getrs<ZView>(st, n, nrhs, ZView((double2 *)A, lda), ZView((double2 *)B, ldb), wk));
    int rc = HPRMAT_OK;
    if (info) {
        HP_CUDA(cudaEventRecord(ev[2], st));
        int h = 0;
        HP_CUDA(cudaMemcpyAsync(&h, info_dev, sizeof(int), cudaMemcpyDeviceToHost, st));
        HP_CUDA(cudaStreamSynchronize(st));
        float ms = 0.f;
        cudaEventElapsedTime(&ms, ev[0], ev[1]);
        info->ms_lu = ms;
        cudaEventElapsedTime(&ms, ev[1], ev[2]);
        info->ms_solve = ms;
        info->ms_total = info->ms_lu + info->ms_solve;
        info->lu_tflops = info->ms_lu > 0 ? (8.0 / 3.0) * (double)n * n * n / (info->ms_lu * 1e-3) * 1e-12 : 0.0;
        if (h != 0) {
            rc = HPRMAT_ESINGULAR;
            info->pivot_index = h;
        }
        info->status = rc;
    }
    return rc;
}
