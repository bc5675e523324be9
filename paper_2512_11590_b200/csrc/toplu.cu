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

// Thread grid of one role: TGI x TGJ threads, thread (ti, tj) owns the elements (ti + TGI a, tj + TGJ b): an RA x RB register
// tile.  8 x 16 threads with 8 x 4 tiles: half the warps of a 16 x 16 grid with 4 x 4 tiles, and the per-column bookkeeping
// (publishing, barrier, operand loads, predicates) is paid per warp -- the kernel is bound by the issue rate of its one SM
// (profiles/r02_toplu.md).
// (profiles/r02_toplu.md).  The complex128 type keeps 16 x 16 threads: two 8 x 4 tiles of double2 do not fit the register file.
constexpr int TGJ = 16;
template <class V> struct TopGrid { static constexpr int TGI = 16; };
template <> struct TopGrid<CView> { static constexpr int TGI = 8; };

// What crosses the roles, double-buffered by column parity
template <class E> struct TopLuSmem {
    E colb[2][TW];   // column j of the partly eliminated block, rows <= j zeroed  (LU role -> LU, XL)
    E rowb[2][TW];   // row j of U, columns <= j zeroed                           (LU role -> LU, Y)
    E xlrow[2][TW];  // row j of XL = inv(L)                                       (XL role -> XL)
    E yrow[2][TW];   // row j of Y = inv(U)^T, not yet scaled by 1/u_jj            (Y role -> Y)
    E ipv[TW];       // 1 / u_jj, from the owner of the diagonal element (formed one column ahead, see the sweep)
};

// 1 / pv = conj(pv) / |pv|^2: the entries of these blocks are O(1) (S = I + coupling-sized terms), so the squared modulus
// cannot overflow; one approximate reciprocal + two Newton steps.  A zero pivot gives zero (reported by the caller).
template <class E> __device__ __forceinline__ E top_pivot_recip(E pv) {
    typedef typename real_of<E>::type T;
    const T den = pv.x * pv.x + pv.y * pv.y;
    T r = den > (T)0 ? rcp_approx(den) : (T)0;
    r = r * ((T)2 - den * r);
    r = r * ((T)2 - den * r);
    return mk(pv.x * r, -pv.y * r);
}

// One CTA factors the w x w block (w <= TW, padded to TW x TW by the identity) WITHOUT interchanges and inverts both
// triangular factors, all out of registers: two groups of threads run three rank-1 sweeps in lock step (the
// factorisation in one group, both inversions in the other),
//   LU:  step j: l_i = a_ij / u_jj (i > j),  a_ic -= l_i u_jc (i, c > j)
//   XL = inv(L):     rows i > j:  XL[i,:] -= l_i XL[j,:]                (row j of XL is final when step j starts)
//   Y  = inv(U)^T = inv(U^T), U^T lower triangular with diagonal u_jj:
//                    Y[j,:] /= u_jj;  rows i > j:  Y[i,:] -= u_ji Y[j,:]   (u_ji = U[j,i]: row j of U, final at step j)
// Column j of L and row j of U are exactly what the LU role publishes at step j, so the two inversions ride one step
// behind the factorisation for free: TW barriers in all instead of 2 TW.
template <class V>
__global__ void __launch_bounds__(2 * TopGrid<V>::TGI * TGJ, 1)
    top_lu_kernel(V A, int w, int c0, int *ipiv, int *info, int *refuted, V dinvL, V dinvU, int *perm, int nbatch) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    constexpr int TGI = TopGrid<V>::TGI;
    constexpr int TL_G = TGI * TGJ;   // threads of one role; two roles advance together, one barrier per column
    constexpr int TL_RA = TW / TGI, TL_RB = TW / TGJ;
    constexpr int TL_CG = TGI < TGJ ? TGI : TGJ;  // columns per compile-time group: j / TGI and j / TGJ are constant inside it
    static_assert(TGJ % TGI == 0 || TGI % TGJ == 0, "one grid dimension divides the other");
    static_assert(TL_G >= TW, "one thread per column writes the interchanges");
    __shared__ TopLuSmem<E> sm;
    const int role = threadIdx.x / TL_G, lt = threadIdx.x % TL_G, ti = lt % TGI, tj = lt / TGI;
    const E zero = mk((T)0, (T)0), one = mk((T)1, (T)0);

    pdl_wait();
    pdl_trigger();
    // LU role: x = the block.  Inversion role: x = XL, y = Y, both start as the identity
    E x[TL_RA][TL_RB], y[TL_RA][TL_RB];
#pragma unroll
    for (int a = 0; a < TL_RA; ++a)
#pragma unroll
        for (int b = 0; b < TL_RB; ++b) {
            const int row = ti + TGI * a, col = tj + TGJ * b;
            x[a][b] = (role == 0 && row < w && col < w) ? A.get(row, col) : (row == col ? one : zero);
            y[a][b] = row == col ? one : zero;
        }
    int bad = 0;
    if (role == 0 && lt == 0) {  // the first pivot's reciprocal; every later one is formed at the end of the step before it
        sm.ipv[0] = top_pivot_recip(x[0][0]);
        if (x[0][0].x == (T)0 && x[0][0].y == (T)0) {
            atomicCAS(info, 0, c0 + 1);
            bad = 1;
        }
    }
    // the column group G is compile-time so that the register tiles are statically indexed: JA = j / TGI, JB = j / TGJ
    static_for<0, TW / TL_CG>([&](auto gc) {
        constexpr int G = decltype(gc)::value;
        constexpr int JA = G * TL_CG / TGI, JB = G * TL_CG / TGJ;
#pragma unroll 1
        for (int jj = 0; jj < TL_CG; ++jj) {
            const int j = TL_CG * G + jj, par = j & 1;
            const int oi = j % TGI, oj = j % TGJ;  // thread coordinates of the owners of row j / column j
            // ---- publish (owners only)
            if (role == 0) {
                if (ti == oi) {  // row j of U; finished columns read as zero
#pragma unroll
                    for (int b = JB; b < TL_RB; ++b) sm.rowb[par][tj + TGJ * b] = (tj + TGJ * b > j) ? x[JA][b] : zero;
                }
                if (tj == oj) {  // column j, not yet divided by the pivot; finished rows read as zero
#pragma unroll
                    for (int a = JA; a < TL_RA; ++a) sm.colb[par][ti + TGI * a] = (ti + TGI * a > j) ? x[a][JB] : zero;
                }
            } else if (ti == oi) {  // rows j of XL and of Y: non-zero in columns <= j only
#pragma unroll
                for (int b = 0; b <= JB; ++b) {
                    sm.xlrow[par][tj + TGJ * b] = x[JA][b];
                    sm.yrow[par][tj + TGJ * b] = y[JA][b];
                }
            }
            __syncthreads();
            const E ip = sm.ipv[j];  // 1 / u_jj
            if (role == 0) {
                // a_ic -= a_ij (u_jc / u_jj): the row is scaled (TL_RB products per thread) rather than the column (TL_RA)
                E cj[TL_RA], u[TL_RB];
#pragma unroll
                for (int a = JA; a < TL_RA; ++a) cj[a] = sm.colb[par][ti + TGI * a];
#pragma unroll
                for (int b = JB; b < TL_RB; ++b) u[b] = cmul_packed(sm.rowb[par][tj + TGJ * b], ip);
#pragma unroll
                for (int a = JA; a < TL_RA; ++a)
#pragma unroll
                    for (int b = JB; b < TL_RB; ++b) x[a][b] = cfnma_packed(x[a][b], cj[a], u[b]);
                // (column j itself is left as a_ij^(j): its u[] entry is zero.  The multipliers l_i = a_ij / u_jj are formed
                // once, after the sweep -- inside it they would be extra work for the one warp every column waits for.)
                // The next pivot u_{j+1,j+1} is final now.  Its reciprocal is formed here, branch-free on every thread's own
                // candidate element so that the chain (reciprocal, two Newton steps) overlaps the update above instead of
                // standing between the next barrier and everybody's first use; the owner publishes it.
                if (j + 1 < TW) {
                    constexpr int GN = G + 1 < TW / TL_CG ? G + 1 : G;
                    constexpr int JAN = GN * TL_CG / TGI, JBN = GN * TL_CG / TGJ;
                    const E pvn = (jj + 1 < TL_CG) ? x[JA][JB] : x[JAN][JBN];
                    const E ipn = top_pivot_recip(pvn);
                    if (ti == (j + 1) % TGI && tj == (j + 1) % TGJ) {
                        sm.ipv[j + 1] = ipn;
                        if (pvn.x == (T)0 && pvn.y == (T)0) {
                            atomicCAS(info, 0, c0 + j + 2);
                            bad = 1;
                        }
                    }
                }
            } else {
                // rows i > j:  XL[i,:] -= l_i XL[j,:]  and  Y[i,:] -= u_ji (Y[j,:] / u_jj);  Y's row j takes its 1/u_jj
                // (l_i = a_ij / u_jj: the 1 / u_jj goes onto row j of XL, JB + 1 products per thread instead of TL_RA)
                E la[TL_RA], ua[TL_RA], xr[TL_RB], yr[TL_RB];
#pragma unroll
                for (int a = JA; a < TL_RA; ++a) {
                    la[a] = sm.colb[par][ti + TGI * a];
                    ua[a] = sm.rowb[par][ti + TGI * a];
                }
#pragma unroll
                for (int b = 0; b <= JB; ++b) {
                    xr[b] = cmul_packed(sm.xlrow[par][tj + TGJ * b], ip);
                    yr[b] = cmul_packed(sm.yrow[par][tj + TGJ * b], ip);
                }
#pragma unroll
                for (int a = JA; a < TL_RA; ++a)
#pragma unroll
                    for (int b = 0; b <= JB; ++b) {
                        x[a][b] = cfnma_packed(x[a][b], la[a], xr[b]);
                        y[a][b] = cfnma_packed(y[a][b], ua[a], yr[b]);
                    }
                if (ti == oi) {
#pragma unroll
                    for (int b = 0; b <= JB; ++b) y[JA][b] = yr[b];
                }
            }
        }
    });
    // ---- results
    if (role == 0) {
#pragma unroll
        for (int b = 0; b < TL_RB; ++b) {
            const int col = tj + TGJ * b;
            const E ipc = sm.ipv[col];  // 1 / u_cc (complete: the last column's barrier has passed)
#pragma unroll
            for (int a = 0; a < TL_RA; ++a) {
                const int row = ti + TGI * a;
                if (row > col) {
                    x[a][b] = cmul_packed(x[a][b], ipc);                   // the multiplier l_row,col
                    if (!(cabs1(x[a][b]) <= (T)0.5)) bad = 1;              // every multiplier, once; also catches NaN
                }
                if (row < w && col < w) A.set(row, col, x[a][b]);
            }
        }
        if (lt < w) ipiv[c0 + lt] = c0 + lt + 1;              // identity interchanges
        if (lt < nbatch) perm[(size_t)lt * PERM_STRIDE] = 0;  // empty swap batches
    } else {
#pragma unroll
        for (int a = 0; a < TL_RA; ++a)
#pragma unroll
            for (int b = 0; b < TL_RB; ++b) {
                const int row = ti + TGI * a, col = tj + TGJ * b;
                if (row < w && col < w) {
                    dinvL.set(row, col, x[a][b]);
                    dinvU.set(col, row, y[a][b]);  // inv(U) = Y^T
                }
            }
    }
    if (__syncthreads_or(bad) && threadIdx.x == 0) atomicAdd(refuted, 1);
}

// counts the multipliers of L (m x w) that violate |l|_1 <= 1/2 (or are NaN): CTA = 256 rows x CHK_C columns
constexpr int CHK_C = 8;
template <class V> __global__ void __launch_bounds__(256) check_multipliers_kernel(V L, int m, int w, int *refuted) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    const int row = blockIdx.x * 256 + threadIdx.x, c0 = blockIdx.y * CHK_C;
    int bad = 0;
    pdl_wait();
    pdl_trigger();
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
    const int b0 = c0 / IB, nbatch = ceil_div(w, IB);
    {
        ProfCat pc(PROF_PANEL);
        const bool prof = prof_enabled();
        if (prof) prof_begin(st, 0.0);
        auto kern = top_lu_kernel<V>;
        HP_CUDA(launch_pdl(kern, dim3(1), dim3(2 * TopGrid<V>::TGI * TGJ), 0, st, A.sub(c0, c0), w, c0, ipiv, info_dev, wk.refuted, dl, du,
                           wk.perm + (size_t)b0 * PERM_STRIDE, nbatch));
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
        if (!wk.accurate && l21_checked(st, m2, w, L21, du, wk.refuted)) return 0;  // complex64: the check rides in the epilogue
        HP_TRY(gemm(st, m2, w, w, 1.0, L21, du, 0.0, L21));
        const bool prof = prof_enabled();
        if (prof) prof_begin(st, 0.0);
        HP_CUDA(launch_pdl(check_multipliers_kernel<V>, dim3(ceil_div(m2, 256), ceil_div(w, CHK_C)), dim3(256), 0, st, L21, m2, w,
                           wk.refuted));
        if (prof) prof_end(st);
        HP_LAUNCHED();
    }
    return 0;
}

template int block_panel<CView>(cudaStream_t, int, CView, int, int, int *, int *, LuWork<CView> &, CView, CView);
template int block_panel<ZView>(cudaStream_t, int, ZView, int, int, int *, int *, LuWork<ZView> &, ZView, ZView);

}  // namespace hp
