// util.cu -- process-wide state behind the C ABI: error strings and the launch counter.
#include <cstdio>
#include <cstdlib>
#include <mutex>
#include <vector>

#include "common.cuh"

namespace hp {
thread_local char g_cuda_err[256] = "";
std::atomic<long long> g_launches{0};
static std::atomic<bool> g_pdl{true};
bool pdl_enabled() { return g_pdl.load(std::memory_order_relaxed); }
static std::atomic<bool> g_lookahead{true};
bool lookahead_enabled() { return g_lookahead.load(std::memory_order_relaxed); }

// ---- optional per-launch timing of the GEMM kernel (bench.py's roofline leg): one CUDA-event pair around every launch
struct ProfRec { cudaEvent_t a, b; double flops; int cat; };
static std::atomic<bool> g_prof_on{false};
static std::mutex g_prof_mu;  // the record below is process-wide (a measurement aid)
thread_local int g_prof_cat = PROF_OTHER;
static double g_cat_ms[PROF_NCAT], g_cat_flops[PROF_NCAT];
static long long g_cat_n[PROF_NCAT];
static std::vector<ProfRec> g_prof;
static std::vector<cudaEvent_t> g_prof_pool;
static cudaEvent_t prof_event() {
    cudaEvent_t e = nullptr;
    if (!g_prof_pool.empty()) { e = g_prof_pool.back(); g_prof_pool.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}
bool prof_enabled() { return g_prof_on; }
void prof_begin(cudaStream_t st, double flops) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    ProfRec r{prof_event(), prof_event(), flops, g_prof_cat};
    cudaEventRecord(r.a, st);
    g_prof.push_back(r);
}
void prof_end(cudaStream_t st) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    cudaEventRecord(g_prof.back().b, st);
}
}  // namespace hp

extern "C" int hprmat_profile(int enable) {
    hp::g_prof_on = enable != 0;
    return HPRMAT_OK;
}
extern "C" int hprmat_profile_read(double *ms, double *flops, long long *launches) {
    double t = 0.0, f = 0.0;
    long long n = 0;
    std::lock_guard<std::mutex> lk(hp::g_prof_mu);
    for (int c = 0; c < hp::PROF_NCAT; ++c) { hp::g_cat_ms[c] = hp::g_cat_flops[c] = 0.0; hp::g_cat_n[c] = 0; }
    for (auto &r : hp::g_prof) {
        if (cudaEventSynchronize(r.b) != cudaSuccess) return HPRMAT_ECUDA;
        float m = 0.f;
        cudaEventElapsedTime(&m, r.a, r.b);
        hp::g_cat_ms[r.cat] += m; hp::g_cat_flops[r.cat] += r.flops; ++hp::g_cat_n[r.cat];
        if (r.flops > 0.0) { t += m; f += r.flops; ++n; }
        hp::g_prof_pool.push_back(r.a);
        hp::g_prof_pool.push_back(r.b);
    }
    hp::g_prof.clear();
    if (ms) *ms = t;
    if (flops) *flops = f;
    if (launches) *launches = n;
    return HPRMAT_OK;
}

extern "C" int hprmat_profile_cat(int cat, double *ms, double *flops, long long *launches) {
    if (cat < 0 || cat >= hp::PROF_NCAT) return -1;
    if (ms) *ms = hp::g_cat_ms[cat];
    if (flops) *flops = hp::g_cat_flops[cat];
    if (launches) *launches = hp::g_cat_n[cat];
    return HPRMAT_OK;
}

extern "C" const char *hprmat_strerror(int code) {
    switch (code) {
        case HPRMAT_OK: return "success";
        case HPRMAT_ESINGULAR: return "matrix is singular (exact zero pivot)";
        case HPRMAT_ENOTCONVERGED: return "iterative refinement did not converge";
        case HPRMAT_ENOMEM: return "out of device memory / workspace too small";
        case HPRMAT_ECUDA: return "CUDA error";
        case HPRMAT_EUNVERIFIED: return "verified-diagonal factorisation refuted or unusable in an unsynchronised call";
        default: return code < 0 ? "invalid argument" : "unknown error";
    }
}
extern "C" const char *hprmat_last_cuda_error(void) { return hp::g_cuda_err; }
extern "C" int hprmat_profile_pdl(int enable) {
    if (enable == 0 || enable == 1) hp::g_pdl.store(enable != 0, std::memory_order_relaxed);
    return hp::pdl_enabled() ? 1 : 0;
}
extern "C" int hprmat_profile_lookahead(int enable) {
    if (enable == 0 || enable == 1) hp::g_lookahead.store(enable != 0, std::memory_order_relaxed);
    return hp::lookahead_enabled() ? 1 : 0;
}
extern "C" long long hprmat_launch_count(void) { return hp::g_launches.load(); }
