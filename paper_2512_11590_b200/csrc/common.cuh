// common.cuh -- shared device/host helpers of the HPRMAT B200 path (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <atomic>

#include "../../include/hprmat.h"

namespace hp {

// ---- error plumbing ------------------------------------------------------------------------------------------------
extern thread_local char g_cuda_err[256];
extern std::atomic<long long> g_launches;

inline int cuda_fail(cudaError_t e, const char *file, int line) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (%s:%d)", cudaGetErrorString(e), file, line);
    return HPRMAT_ECUDA;
}
#define HP_CUDA(x)                                                   \
    do {                                                             \
        cudaError_t e__ = (x);                                       \
        if (e__ != cudaSuccess) return hp::cuda_fail(e__, __FILE__, __LINE__); \
    } while (0)
#define HP_TRY(x)                 \
    do {                          \
        int r__ = (x);            \
        if (r__ != 0) return r__; \
    } while (0)
// after a kernel launch: count it and pick up launch-configuration errors
#define HP_LAUNCHED()                  \
    do {                               \
        hp::g_launches.fetch_add(1, std::memory_order_relaxed); \
        HP_CUDA(cudaPeekAtLastError()); \
    } while (0)

constexpr int kNumSMs = 148;  // B200

// launch categories of the per-launch timing (hprmat_profile_cat)
enum { PROF_LU_GEMM = 0, PROF_LU_TRSM = 1, PROF_PANEL = 2, PROF_LASWP = 3, PROF_SOLVE = 4, PROF_OTHER = 5, PROF_NCAT = 6 };
extern thread_local int g_prof_cat;
struct ProfCat {  // RAII: category of the launches issued in this scope
    int prev;
    explicit ProfCat(int c) : prev(g_prof_cat) { g_prof_cat = c; }
    ~ProfCat() { g_prof_cat = prev; }
};
bool prof_enabled();
void prof_begin(cudaStream_t st, double flops);
void prof_end(cudaStream_t st);

// Grouped ("super-tile") CTA rasterisation of a tiles_m x tiles_n grid: consecutive CTA ids walk down GROUP tile rows, then
// step one tile column, so that the ~148 CTAs in flight cover a roughly square block of C and share their A and B panels
// through L2 instead of streaming the whole of A once per tile column.
__device__ __forceinline__ void raster(int pid, int tiles_m, int tiles_n, int group, int &tm, int &tn) {
    const int per_group = group * tiles_n;
    const int gid = pid / per_group;
    const int first = gid * group;
    const int gsz = min(tiles_m - first, group);
    const int r = pid - gid * per_group;
    tm = first + r % gsz;
    tn = r / gsz;
}

// Lazy, thread-safe, per-device configuration of a kernel's dynamic shared-memory limit (cudaFuncSetAttribute is per
// device; setting it twice is harmless, so the only shared state is a monotone per-device maximum).
struct SmemCfg {
    std::atomic<int> bytes[32];
};
template <class K> inline int configure_smem(SmemCfg &c, K kern, size_t bytes) {
    int dev = 0;
    HP_CUDA(cudaGetDevice(&dev));
    const bool tracked = dev >= 0 && dev < 32;
    if (tracked && c.bytes[dev].load(std::memory_order_acquire) >= (int)bytes) return 0;
    HP_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    if (tracked) {
        int cur = c.bytes[dev].load(std::memory_order_relaxed);
        while (cur < (int)bytes && !c.bytes[dev].compare_exchange_weak(cur, (int)bytes, std::memory_order_release)) {
        }
    }
    return 0;
}

// Programmatic dependent launch (PDL): a kernel launched through launch_pdl may become resident while its predecessor on
// the stream is still running, do its prologue (barrier init, TMEM allocation, descriptor prefetch) and then MUST execute
// pdl_wait() -- in every CTA, before its first access to global memory -- which returns once the predecessor grid has
// completed and its writes are visible.  pdl_trigger() lets the NEXT launch start that early.  The LU issues thousands of
// small dependent kernels; this hides their launch latency and prologues behind the predecessor's tail.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;\n" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory"); }
#endif
bool pdl_enabled();  // util.cu (hprmat_profile_pdl)
bool lookahead_enabled();  // util.cu (hprmat_profile_lookahead)
template <class... KArgs, class... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t lc = {};
    lc.gridDim = grid;
    lc.blockDim = block;
    lc.dynamicSmemBytes = smem;
    lc.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = at;
    lc.numAttrs = pdl_enabled() ? 1 : 0;
    return cudaLaunchKernelEx(&lc, kern, KArgs(args)...);
}

// Real decomposition of the complex128 GEMM (3 = 3M, 4 = 4M) in force on this host thread: the process default
// (hprmat_zgemm_algo) unless a context's own setting is installed for the duration of one of its calls.
int zgemm_algo_in_force();
struct ScopedZgemmAlgo {
    int prev;
    explicit ScopedZgemmAlgo(int algo);
    ~ScopedZgemmAlgo();
};

int sm_reserve_in_force();  // cgemm2.cu
struct ScopedSmReserve {
    int prev;
    explicit ScopedSmReserve(int sms);
    ~ScopedSmReserve();
};
int cgemm_variant_in_force();  // cgemm.cu (measurement aid: which tcgen05 kernel serves the planar complex64 GEMM)

inline int ceil_div(long a, long b) { return (int)((a + b - 1) / b); }
inline long round_up(long a, long b) { return (a + b - 1) / b * b; }

// ---- complex matrix views ------------------------------------------------------------------------------------------
// The FP64 path stores interleaved complex128 (LAPACK layout; the raw solve factorises the caller's array in place).
// The mixed path stores SPLIT (planar) complex64 -- one float plane for the real and one for the imaginary part -- so
// that the trailing update is four real TF32 tensor-core products on operands that can be fed to the MMA unchanged.
struct ZView {
    typedef double real_t;
    typedef double2 elem_t;
    double2 *p;
    long ld;
    __host__ __device__ ZView() : p(nullptr), ld(0) {}
    __host__ __device__ ZView(double2 *p_, long ld_) : p(p_), ld(ld_) {}
    __host__ __device__ ZView sub(long i, long j) const { return ZView(p + j * ld + i, ld); }
    __device__ __forceinline__ double2 get(long i, long j) const { return p[j * ld + i]; }
    __device__ __forceinline__ void set(long i, long j, double2 v) const { p[j * ld + i] = v; }
};

struct CView {
    typedef float real_t;
    typedef float2 elem_t;
    float *re, *im;
    long ld;
    __host__ __device__ CView() : re(nullptr), im(nullptr), ld(0) {}
    __host__ __device__ CView(float *r_, float *i_, long ld_) : re(r_), im(i_), ld(ld_) {}
    __host__ __device__ CView sub(long i, long j) const { return CView(re + j * ld + i, im + j * ld + i, ld); }
    __device__ __forceinline__ float2 get(long i, long j) const {
        return make_float2(re[j * ld + i], im[j * ld + i]);
    }
    __device__ __forceinline__ void set(long i, long j, float2 v) const {
        re[j * ld + i] = v.x;
        im[j * ld + i] = v.y;
    }
};

// ---- complex arithmetic on double2 / float2 -------------------------------------------------------------------------
template <class E> struct real_of;
template <> struct real_of<double2> { typedef double type; };
template <> struct real_of<float2> { typedef float type; };

__device__ __forceinline__ double2 mk(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 mk(float a, float b) { return make_float2(a, b); }

template <class E> __device__ __forceinline__ E cmul(E a, E b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <class E> __device__ __forceinline__ E cadd(E a, E b) { return mk(a.x + b.x, a.y + b.y); }
template <class E> __device__ __forceinline__ E csub(E a, E b) { return mk(a.x - b.x, a.y - b.y); }
// a - b*c
template <class E> __device__ __forceinline__ E cfnma(E a, E b, E c) {
    typedef typename real_of<E>::type T;
    T re = a.x - b.x * c.x;
    re = re + b.y * c.y;
    T im = a.y - b.x * c.y;
    im = im - b.y * c.x;
    return mk(re, im);
}
template <class E> __device__ __forceinline__ typename real_of<E>::type cabs1(E a) { return fabs(a.x) + fabs(a.y); }
// 1/a with scaling against overflow (Smith)
template <class E> __device__ __forceinline__ E crecip(E a) {
    typedef typename real_of<E>::type T;
    if (fabs(a.x) >= fabs(a.y)) {
        T r = a.y / a.x, d = a.x + a.y * r;
        return mk((T)1 / d, -r / d);
    } else {
        T r = a.x / a.y, d = a.x * r + a.y;
        return mk(r / d, (T)-1 / d);
    }
}

// 1/a by Smith's formula on the reciprocal intrinsics (two dependent reciprocals, no IEEE-division slow paths)
__device__ __forceinline__ float rcp_rn(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double rcp_rn(double x) { return __drcp_rn(x); }
// approximate reciprocal (to be refined by Newton steps)
__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ double rcp_approx(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    return r;
}
template <class E> __device__ __forceinline__ E crecip_fast(E a) {
    typedef typename real_of<E>::type T;
    if (fabs(a.x) >= fabs(a.y)) {
        const T r = a.y * rcp_rn(a.x), id = rcp_rn(a.x + a.y * r);
        return mk(id, -r * id);
    } else {
        const T r = a.x * rcp_rn(a.y), id = rcp_rn(a.x * r + a.y);
        return mk(r * id, -id);
    }
}

// Packed FP32 pairs (Blackwell FFMA2: one instruction, two lanes): complex64 arithmetic at half the FP32 issue count.
// a - b*c  and  a*b  for float2, same rounding as the scalar forms up to the fused multiply-adds.
__device__ __forceinline__ unsigned long long f2_pack(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float2 f2_unpack(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ unsigned long long f2_fma(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long f2_mul(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float2 cfnma_packed(float2 a, float2 b, float2 c) {
    unsigned long long acc = f2_fma(f2_pack(-b.x, -b.x), f2_pack(c.x, c.y), f2_pack(a.x, a.y));
    acc = f2_fma(f2_pack(b.y, -b.y), f2_pack(c.y, c.x), acc);
    return f2_unpack(acc);
}
__device__ __forceinline__ double2 cfnma_packed(double2 a, double2 b, double2 c) { return cfnma(a, b, c); }
__device__ __forceinline__ float2 cmul_packed(float2 a, float2 b) {
    unsigned long long acc = f2_mul(f2_pack(a.x, a.x), f2_pack(b.x, b.y));
    acc = f2_fma(f2_pack(-a.y, a.y), f2_pack(b.y, b.x), acc);
    return f2_unpack(acc);
}
__device__ __forceinline__ double2 cmul_packed(double2 a, double2 b) { return cmul(a, b); }

// compile-time loop: f(IntC<I>) for I = B .. E-1 (keeps register-resident tiles statically indexed)
template <int I> struct IntC { static constexpr int value = I; };
template <int B, int E_, class F> __device__ __forceinline__ void static_for(F &&f) {
    if constexpr (B < E_) {
        f(IntC<B>{});
        static_for<B + 1, E_>(f);
    }
}

}  // namespace hp
