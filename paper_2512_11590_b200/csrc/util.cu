// util.cu -- process-wide state behind the C ABI: error strings and the launch counter.
#include "common.cuh"

namespace hp {
thread_local char g_cuda_err[256] = "";
long long g_launches = 0;
}  // namespace hp

extern "C" const char *hprmat_strerror(int code) {
    switch (code) {
        case HPRMAT_OK: return "success";
        case HPRMAT_ESINGULAR: return "matrix is singular (exact zero pivot)";
        case HPRMAT_ENOTCONVERGED: return "iterative refinement did not converge";
        case HPRMAT_ENOMEM: return "out of device memory / workspace too small";
        case HPRMAT_ECUDA: return "CUDA error";
        default: return code < 0 ? "invalid argument" : "unknown error";
    }
}
extern "C" const char *hprmat_last_cuda_error(void) { return hp::g_cuda_err; }
extern "C" long long hprmat_launch_count(void) { return hp::g_launches; }
