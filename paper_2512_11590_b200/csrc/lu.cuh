// lu.cuh -- blocked recursive LU with partial pivoting and the triangular solves, for both matrix views.
#pragma once
#include "common.cuh"

namespace hp {

constexpr int IB = 32;        // panel width = swap batch = smallest inverted diagonal block
constexpr int LEAF = 128;     // largest inverted diagonal block = leaf of the triangular-solve recursion (one GEMM M tile,
                              // so that the leaf product B <- inv * B may run in place)
constexpr int NLEV = 3;       // inverted diagonal blocks are kept at sizes IB << lev, lev = 0 .. NLEV-1
// "Solve block": the full inverses of the SB x SB diagonal blocks of L and U are kept as well, so that a triangular solve is
// N/SB dependent steps of large dense GEMMs instead of N/LEAF.  Per type, by measurement at configs[3]: the complex64 solves
// are a chain of latency-bound launches (2048: first solve 6.4 -> 4.2 ms, a refinement step 7.9 -> 6.0 ms, the factorisation
// pays 2 ms for the larger inverses); the complex128 ones are flop bound and the larger inverses cost the LU more than the
// solves gain (1024).
template <class V> struct SolveBlock { static constexpr int value = 1024; };
template <> struct SolveBlock<CView> { static constexpr int value = 2048; };
constexpr int MAXG = kNumSMs; // CTAs of the cooperative panel kernel (one per SM)
constexpr int LA_MIN_N = 4096;  // smallest matrix whose factorisation looks ahead (LuWork::la_*)
constexpr int LA_SM_RESERVE = 40;  // SMs the deferred update's persistent GEMMs leave to the panel chain (8 .. 64 measured:
                                  // 117.8, 117.1, 116.1, 116.5, 114.4, 115.0, 116.5 ms per step at configs[3]; off: 120.3)
constexpr int LA_MAX_W = 32768;   // widest node that looks ahead: beyond, the deferred GEMM is so long that running it on 108 SMs
                                  // costs more than the overlap returns (configs[4] root, w = 51200: +17 ms; below: neutral there,
                                  // -3.4 ms at configs[3]).  complex64 only: the FP64 GEMMs are not persistent and gain nothing.
constexpr int LA_MIN_COLS = 512; // smallest deferred column range worth a fork / join
constexpr int TW = 64;        // width of the block panel of a factorisation with verified diagonal pivots (toplu.cu): its top
                              // block is factored and inverted by one CTA out of registers and shared memory

// GEMM back-ends (zgemm.cu / cgemm.cu): C <- beta*C + alpha*A*B.  nbatch > 1: operand b lives at view + b*stride
// elements.  C may alias B when m <= 128 (a single M tile of the kernel that is chosen then) and beta == 0: the in-place
// leaf product B <- inv * B of the triangular solves (lu.cu).
int gemm(cudaStream_t st, int m, int n, int k, double alpha, ZView A, ZView B, double beta, ZView C);
int gemm(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C);
// persistent tcgen05 kernel behind gemm(CView) (cgemm2.cu); shape: 0 = single CTAs (128 x 128 tiles), 1 / 2 = CTA pairs, cta_group::2 (256 x 128 / 256 x 256 tiles).  chk_count != nullptr: the
// epilogue also counts results with |re| + |im| > chk_thr.  C may alias A when n <= 128, B when m <= 128 (pair == false).
// wave_ctr: 256 device words of scratch owned by the caller for the duration of the launch (null: no wave barrier)
int cgemm2(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, int shape, float chk_thr = 0.f,
           int *chk_count = nullptr, unsigned *wave_ctr = nullptr);
// gemm(CView) with the wave-barrier scratch of a factorisation's workspace
int cgemm_ws(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, unsigned *wave_ctr);
// few output tiles, deep K: every 128 x 128 tile by a cluster of `slices` (2, 4, 8) CTAs along K, deterministic reduction through
// distributed shared memory (cgemm_splitk.cu).  C must not alias A or B.
int cgemm_splitk(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C, int slices);
// FP32-class accuracy variant for the planar complex64 type (3xTF32, cgemm3.cu); C may alias B when m <= 128, beta == 0
int cgemm3(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C);
// tcgen05 version (cgemm3x.cu; C distinct from A and B) and the dispatcher between the two
int cgemm3x(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C);
int cgemm3_any(cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C);
int cgemm3_batched(cudaStream_t st, int m, int n, int k, double alpha, CView A, long strideA, CView B, long strideB, double beta,
                   CView C, long strideC, int nbatch);
int zgemm_batched(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, long strideA,
                  const double2 *B, long ldb, long strideB, double beta, double2 *C, long ldc, long strideC, int nbatch);

// Workspace of one factorisation (device memory carved from a caller-provided buffer).
template <class V> struct LuWork {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    int n = 0, nblk = 0;
    V dinvL[NLEV], dinvU[NLEV];  // level lev: blocks of s x s, s = IB << lev, block b at column offset b*s, ld = s:
                                 // inverses of the unit-lower / upper triangle of the diagonal block at (b*s, b*s)
    V binvL, binvU;      // inverses of the SB-aligned diagonal blocks (of size min(SB, n - b SB) > LEAF), ld = sbld, block b at
                         // column offset b*sbld; for the complex64 type getrf leaves their LEAF-diagonal blocks zeroed
                         // (the solves apply those from dinvL/dinvU[NLEV-1] with the 3xTF32 kernel)
    V tmp;               // sbld x tmp_cols scratch: out-of-place leaf product
    long tmp_cols = 0;   // = max(n, 256) for the workspace's own scratch
    long sbld = 0;
    // Look-ahead of the factorisations WITHOUT interchanges (speculate): at a node of the recursion the update of the columns the
    // right child does not need yet (everything right of ITS left child) runs on another stream, under the factorisation of that
    // left child, whose chains of small dependent kernels leave most SMs idle.  Nested NLA deep: one stream, one event pair and
    // one scratch per level (device scratch: carve; host resources: set by the owner of the workspace, null = no look-ahead).
    static constexpr int NLA = 3;
    V la_tmp[NLA];       // sbld x la_cols each (n >= LA_MIN_N only)
    long la_cols = 0;
    cudaStream_t la_stream[NLA] = {nullptr, nullptr, nullptr};
    cudaEvent_t la_fork[NLA] = {nullptr, nullptr, nullptr}, la_join[NLA] = {nullptr, nullptr, nullptr};
    int wave_base = 0, wave_mask = 7;  // this (copy of the) workspace's share of the wave-barrier slots
    unsigned *wave_sync = nullptr;  // (8 + 4 NLA) x 256 words: wave-barrier counters of the persistent complex64 GEMM (cgemm2.cu), one
    int wave_next = 0;              // slot per deep trailing update in flight (host-side round robin)
    int *refuted = nullptr;    // device counter: multipliers that refuted the diagonal-pivot speculation (toplu.cu); zeroed by getrf
    bool speculate = false;    // host-side: the matrix is expected to pivot on its diagonal (S = K_d^-1 (C - E I)): factor
                               // without interchanges and VERIFY (toplu.cu); the caller checks *refuted afterwards
    bool accurate = false;     // host-side, complex64 only: EVERY product of the factorisation and of the solves in FP32-class
                               // arithmetic (3xTF32) instead of single-pass TF32 -- general matrices whose condition number
                               // is beyond 2^11 (raw mixed solve after a failed refinement; the literal Type-3 Schur matrix)
    bool side_used = false; // host-side: something of this factorisation was enqueued on the side stream
    // host-side resources for the side stream (kept block inverses are built under the factorisation).  A context sets its
    // own (hprmat_setup); when null, a per-device pool serves the raw entries (lu.cu)
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    bool use_big = true; // host-side switch: off while an SB inverse is being built from the LEAF-level recursion
    int *perm = nullptr; // nblk x (1 + 4*IB): count, dst rows[2*IB], src rows[2*IB]  (net permutation of each swap batch)
    T *cand_val = nullptr;
    int *cand_row = nullptr;
    E *cand_data = nullptr, *jrow = nullptr;
    unsigned *counter = nullptr;
    unsigned bar_base = 0; // host-side running value of the grid-barrier counter
    unsigned long long *slots = nullptr; // epoch-tagged exchange words of the register-resident panel kernel (lu.cu)
    unsigned ep_base = 0;  // host-side running column count (epoch base) of that kernel
    // look_ahead: also carve the scratch of the look-ahead levels (la_tmp; contexts' complex64 workspace only)
    static size_t bytes(int n, bool look_ahead = false);
    // carve from p (must be 256-byte aligned); returns bytes used
    size_t carve(void *p, int n, bool look_ahead = false);
};

constexpr int PERM_STRIDE = 1 + 4 * IB;

// A = P L U in place (Eq. 5).  ipiv: device, 1-based LAPACK interchanges.  info_dev: device int, set to
// the first zero pivot (1-based) or left 0 (caller zeroes it).
template <class V> int getrf(cudaStream_t st, int n, V A, int *ipiv, int *info_dev, LuWork<V> &w);
// B <- A^-1 B with the factors (forward and backward substitution).
template <class V> int getrs(cudaStream_t st, int n, int nrhs, V A, V B, LuWork<V> &w);

}  // namespace hp
