// toplu.cu -- the "block panel" of the factorisations with VERIFIED DIAGONAL PIVOTS (Eq. 5: LU with
// partial pivoting; :153-190 Eqs. 7-9: the block-preconditioned matrix S = K_d^-1 (C - E I) = I + coupling-sized entries).
//
// Partial pivoting picks, in column j, the first row of maximal |re| + |im| among rows >= j of the partly eliminated column,
// i.e. among the candidates a_ij^(j) = l_ij u_jj.  When that is the diagonal in every column the panel needs no search and no
// interchange, and a TW-column panel of height m factors as
//     top block  A11 = L11 U11          (one CTA, this file: registers + shared memory, no pivot search),
//     L21 = A21 U11^-1                  (one tensor-core GEMM with the inverse of U11 that the top-block kernel also emits),
// The speculation is VERIFIED, not assumed: |l_ij|_1 <= 1/2 for every multiplier (top block: in the kernel; L21: a check
// pass over the GEMM's output) implies |a_ij^(j)|_1 <= sqrt(2) |l_ij|_1 |u_jj|_1 < |u_jj|_1, so the diagonal IS partial
// pivoting's choice, with margin against the rounding differences between this operation order and the column-by-column
// one.  Any violation (or a zero pivot) is counted in *refuted; the callers (ctx.cu) then redo the factorisation with the
// pivoting panels of panel.cu.  For S of the BASELINE configs max |l_ij| is ~5e-3.
//
// The kernel also emits the inverses of the unit-lower and upper triangles of the top block (the leaves of the triangular-
// solve recursion of lu.cu), the identity interchanges and empty swap batches.
#include "lu.cuh"

namespace hp {

namespace {

constexpr int TL_NT = 256;   // 16 x 16 threads; thread (ti, tj) owns the elements (ti + 16 a, tj + 16 b), a, b = 0..3
constexpr int TL_R = TW / 16;

template <class E> struct TopLuSmem {
    E tile[TW * TW];         // column-major, ld = TW: the factored top block
    E rowb[2][2][TW];        // [which sweep][parity][col]: the row every thread needs in a step
    E colb[2][TW];           // [parity][row]: column j of the LU sweep
    E invp[TW];              // 1 / u_jj (0 for a zero pivot), published by the owner of the diagonal element
};

template <class V>
__global__ void __launch_bounds__(TL_NT, 1)
    top_lu_kernel(V A, int w, int c0, int *ipiv, int *info, int *refuted, V dinvL, V dinvU, int *perm, int nbatch) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    extern __shared__ __align__(16) unsigned char smraw[];
    TopLuSmem<E> &sm = *reinterpret_cast<TopLuSmem<E> *>(smraw);
    const int tid = threadIdx.x, ti = tid & 15, tj = tid >> 4;
    const E zero = mk((T)0, (T)0), one = mk((T)1, (T)0);

    // ---- the block, padded to TW x TW by the identity, in registers
    E x[TL_R][TL_R];
#pragma unroll
    for (int a = 0; a < TL_R; ++a)
#pragma unroll
        for (int b = 0; b < TL_R; ++b) {
            const int row = ti + 16 * a, col = tj + 16 * b;
            x[a][b] = (row < w && col < w) ? A.get(row, col) : (row == col ? one : zero);
        }
    int bad = 0;
    // ---- LU without interchanges, one rank-1 update per step; JB = j / 16 is compile-time so that the register tile is
    //      statically indexed; rows / columns of tile index < JB are finished
    static_for<0, TL_R>([&](auto jbc) {
        constexpr int JB = decltype(jbc)::value;
#pragma unroll 1
        for (int jj = 0; jj < 16; ++jj) {
            const int j = 16 * JB + jj, par = j & 1;
            if (ti == jj) {
#pragma unroll
                for (int b = JB; b < TL_R; ++b) sm.rowb[0][par][tj + 16 * b] = x[JB][b];
            }
            if (tj == jj) {
#pragma unroll
                for (int a = JB; a < TL_R; ++a) sm.colb[par][ti + 16 * a] = x[a][JB];
                if (ti == jj) {  // the pivot's owner inverts it once for everybody (the long-latency part of the step)
                    const E pv = x[JB][JB];
                    const bool sing = (pv.x == (T)0 && pv.y == (T)0);
                    sm.invp[j] = sing ? zero : crecip_fast(pv);
                    if (sing) {
                        atomicCAS(info, 0, c0 + j + 1);
                        bad = 1;
                    }
                }
            }
            __syncthreads();
            const E ip = sm.invp[j];
            E l[TL_R], u[TL_R];
#pragma unroll
            for (int a = JB; a < TL_R; ++a) {
                const int row = ti + 16 * a;
                l[a] = row > j ? cmul(sm.colb[par][row], ip) : zero;
                if (!(cabs1(l[a]) <= (T)0.5)) bad = 1;  // also catches NaN
            }
#pragma unroll
            for (int b = JB; b < TL_R; ++b) {
                const int col = tj + 16 * b;
                u[b] = col > j ? sm.rowb[0][par][col] : zero;
            }
#pragma unroll
            for (int a = JB; a < TL_R; ++a)
#pragma unroll
                for (int b = JB; b < TL_R; ++b) x[a][b] = cfnma(x[a][b], l[a], u[b]);
            if (tj == jj) {
#pragma unroll
                for (int a = JB; a < TL_R; ++a)
                    if (ti + 16 * a > j) x[a][JB] = l[a];
            }
        }
    });
    // ---- factored block to shared memory (operand of the two inversion sweeps) and back to the matrix
#pragma unroll
    for (int a = 0; a < TL_R; ++a)
#pragma unroll
        for (int b = 0; b < TL_R; ++b) {
            const int row = ti + 16 * a, col = tj + 16 * b;
            sm.tile[col * TW + row] = x[a][b];
            if (row < w && col < w) A.set(row, col, x[a][b]);
        }
    if (tid < w) ipiv[c0 + tid] = c0 + tid + 1;      // identity interchanges
    if (tid < nbatch) perm[(size_t)tid * PERM_STRIDE] = 0;  // empty swap batches
    if (__syncthreads_or(bad) && tid == 0) atomicAdd(refuted, 1);

    // ---- inverses of the unit-lower triangle L and of the upper triangle U, both by rank-1 sweeps on the identity:
    //        XL: for j ascending:   rows i > j:  XL[i,:] -= L[i,j] XL[j,:]      (row j is final when it is used)
    //        XU: for j descending:  XU[j,:] /= u_jj;  rows i < j:  XU[i,:] -= U[i,j] XU[j,:]
    //      Step s does column j = s of L and column j = TW-1-s of U, so that one barrier serves both.
    E xl[TL_R][TL_R], xu[TL_R][TL_R];
#pragma unroll
    for (int a = 0; a < TL_R; ++a)
#pragma unroll
        for (int b = 0; b < TL_R; ++b) xl[a][b] = xu[a][b] = (ti + 16 * a == tj + 16 * b) ? one : zero;
    static_for<0, TL_R>([&](auto jbc) {
        constexpr int JB = decltype(jbc)::value;  // block of the L column; the U column is in block TL_R-1-JB
        constexpr int UB = TL_R - 1 - JB;
#pragma unroll 1
        for (int jj = 0; jj < 16; ++jj) {
            const int jl = 16 * JB + jj, ju = TW - 1 - jl, par = jj & 1;
            if (ti == jj) {  // row jl of XL: non-zero in columns <= jl
#pragma unroll
                for (int b = 0; b <= JB; ++b) sm.rowb[0][par][tj + 16 * b] = xl[JB][b];
            }
            if (ti == 15 - jj) {  // row ju of XU, scaled by 1/u_jj: non-zero in columns >= ju
                const E ipu = sm.invp[ju];
#pragma unroll
                for (int b = UB; b < TL_R; ++b) {
                    xu[UB][b] = cmul(xu[UB][b], ipu);
                    sm.rowb[1][par][tj + 16 * b] = xu[UB][b];
                }
            }
            __syncthreads();
            {
                E l[TL_R], r[TL_R];
#pragma unroll
                for (int a = JB; a < TL_R; ++a) {
                    const int row = ti + 16 * a;
                    l[a] = row > jl ? sm.tile[jl * TW + row] : zero;
                }
#pragma unroll
                for (int b = 0; b <= JB; ++b) {
                    const int col = tj + 16 * b;
                    r[b] = col <= jl ? sm.rowb[0][par][col] : zero;
                }
#pragma unroll
                for (int a = JB; a < TL_R; ++a)
#pragma unroll
                    for (int b = 0; b <= JB; ++b) xl[a][b] = cfnma(xl[a][b], l[a], r[b]);
            }
            {
                E uu[TL_R], r[TL_R];
#pragma unroll
                for (int a = 0; a <= UB; ++a) {
                    const int row = ti + 16 * a;
                    uu[a] = row < ju ? sm.tile[ju * TW + row] : zero;
                }
#pragma unroll
                for (int b = UB; b < TL_R; ++b) {
                    const int col = tj + 16 * b;
                    r[b] = col >= ju ? sm.rowb[1][par][col] : zero;
                }
#pragma unroll
                for (int a = 0; a <= UB; ++a)
#pragma unroll
                    for (int b = UB; b < TL_R; ++b) xu[a][b] = cfnma(xu[a][b], uu[a], r[b]);
            }
        }
    });
#pragma unroll
    for (int a = 0; a < TL_R; ++a)
#pragma unroll
        for (int b = 0; b < TL_R; ++b) {
            const int row = ti + 16 * a, col = tj + 16 * b;
            if (row < w && col < w) {
                dinvL.set(row, col, xl[a][b]);
                dinvU.set(row, col, xu[a][b]);
            }
        }
}

// counts the multipliers of L (m x w) that violate |l|_1 <= 1/2 (or are NaN): CTA = 256 rows x CHK_C columns
constexpr int CHK_C = 8;
template <class V> __global__ void __launch_bounds__(256) check_multipliers_kernel(V L, int m, int w, int *refuted) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    const int row = blockIdx.x * 256 + threadIdx.x, c0 = blockIdx.y * CHK_C;
    int bad = 0;
    if (row < m) {
        E v[CHK_C];
#pragma unroll
        for (int c = 0; c < CHK_C; ++c) v[c] = c0 + c < w ? L.get(row, c0 + c) : mk((T)0, (T)0);
#pragma unroll
        for (int c = 0; c < CHK_C; ++c)
            if (!(cabs1(v[c]) <= (T)0.5)) bad = 1;
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicAdd(refuted, 1);
}

}  // namespace

// L21 <- L21 U11^-1 with the multiplier check fused into the GEMM's epilogue: the persistent tcgen05 kernel only
static bool l21_checked(cudaStream_t, int, int, ZView, ZView, int *) { return false; }
static bool l21_checked(cudaStream_t st, int m2, int w, CView L21, CView du, int *refuted) {
    if (cgemm_variant_in_force() == 1) return false;
    const bool prof = prof_enabled();
    if (prof) prof_begin(st, 8.0 * m2 * w * w);
    const int rc = cgemm2(st, m2, w, w, 1.0, L21, du, 0.0, L21, m2 > 128 ? 1 : 0, 0.5f, refuted);
    if (prof) prof_end(st);
    return rc == 0;
}

template <class V> int block_panel(cudaStream_t st, int n, V A, int c0, int w, int *ipiv, int *info_dev, LuWork<V> &wk, V dl, V du) {
    typedef typename V::elem_t E;
    const size_t smem = sizeof(TopLuSmem<E>);
    auto kern = top_lu_kernel<V>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, smem));
    const int b0 = c0 / IB, nbatch = ceil_div(w, IB);
    {
        ProfCat pc(PROF_PANEL);
        const bool prof = prof_enabled();
        if (prof) prof_begin(st, 0.0);
        kern<<<1, TL_NT, smem, st>>>(A.sub(c0, c0), w, c0, ipiv, info_dev, wk.refuted, dl, du, wk.perm + (size_t)b0 * PERM_STRIDE,
                                     nbatch);
        if (prof) prof_end(st);
        HP_LAUNCHED();
    }
    const int m2 = n - c0 - w;
    if (m2 <= 0) return 0;
    // L21 = A21 U11^-1, in place: every CTA of the GEMM reads its own rows of A21 (all w columns) before it writes them
    // (w <= one N tile of either GEMM kernel)
    V L21 = A.sub(c0 + w, c0);
    {
        ProfCat pc(PROF_PANEL);
        if (l21_checked(st, m2, w, L21, du, wk.refuted)) return 0;  // complex64: the check rides in the GEMM's epilogue
        HP_TRY(gemm(st, m2, w, w, 1.0, L21, du, 0.0, L21));
        const bool prof = prof_enabled();
        if (prof) prof_begin(st, 0.0);
        check_multipliers_kernel<V><<<dim3(ceil_div(m2, 256), ceil_div(w, CHK_C)), 256, 0, st>>>(L21, m2, w, wk.refuted);
        if (prof) prof_end(st);
        HP_LAUNCHED();
    }
    return 0;
}

template int block_panel<CView>(cudaStream_t, int, CView, int, int, int *, int *, LuWork<CView> &, CView, CView);
template int block_panel<ZView>(cudaStream_t, int, ZView, int, int, int *, int *, LuWork<ZView> &, ZView, ZView);

}  // namespace hp
