// api_raw.cu -- raw dense complex entries of the C ABI: LU, triangular solves, workspace query (FP64 part).
// PAPER.md:119 ("all solvers take the matrix M and right-hand side b and return c"), :125-137 (ZGESV semantics).
#include "lu.cuh"

using namespace hp;

namespace hp {
size_t raw_workspace_fp64(int n) { return LuWork<ZView>::bytes(n) + 256; }
}  // namespace hp

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
