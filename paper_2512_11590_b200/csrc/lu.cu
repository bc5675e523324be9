// lu.cu -- recursive blocked LU with partial pivoting, M = P L U (Eq. 5), and the triangular
// solves for the nch right-hand sides (PAPER.md:127 "forward and backward substitution"; :137 step 3).
//
// Structure:
//   getrf_rec(c0,c1): width <= IB -> panel kernel (panel.cu); else factor the left half, U12 <- L11^-1 A12 (recursive TRSM
//   whose leaves multiply by kept inverses of the diagonal blocks), A22 <- A22 - L21 U12 (tensor-core GEMM), factor the
//   right half.  All O(N^3) work is GEMM with K up to N/2, so the trailing update is compute- not HBM-bound.
//   Kept inverses: IB x IB from the panel kernel, doubled up to LEAF = 128 (inv_double_kernel), and the full inverses of
//   the SB = 1024 diagonal blocks ("solve blocks"), so that a triangular solve is N/SB dependent steps of large GEMMs.
//   Row interchanges: right after each panel, its IB swaps are folded into one net permutation of <= 2 IB rows and
//   applied to ALL other columns of the matrix by a gather/scatter kernel (independent loads, no swap chain).
#include "lu.cuh"
#include "panel.cuh"

#include <algorithm>
#include <mutex>

namespace hp {

// ------------------------------------------------------------------------------------------------- workspace
template <class V> static V alloc_view(char *&p, long rows, long cols);
template <> ZView alloc_view<ZView>(char *&p, long rows, long cols) {
    ZView v((double2 *)p, rows);
    p += round_up(rows * cols * sizeof(double2), 256);
    return v;
}
template <> CView alloc_view<CView>(char *&p, long rows, long cols) {
    float *re = (float *)p;
    p += round_up(rows * cols * sizeof(float), 256);
    float *im = (float *)p;
    p += round_up(rows * cols * sizeof(float), 256);
    return CView(re, im, rows);
}

template <class V> size_t LuWork<V>::carve(void *base, int n_, bool look_ahead) {
    char *p = (char *)base;
    n = n_;
    nblk = ceil_div(n, IB);
    auto take = [&](size_t bytes) {
        char *q = p;
        p += round_up((long)bytes, 256);
        return q;
    };
    for (int lev = 0; lev < NLEV; ++lev) {
        const long sz = (long)IB << lev;
        dinvL[lev] = alloc_view<V>(p, sz, (long)ceil_div(n, sz) * sz);
        dinvU[lev] = alloc_view<V>(p, sz, (long)ceil_div(n, sz) * sz);
    }
    constexpr int SB = SolveBlock<V>::value;
    sbld = std::min<long>(SB, round_up(std::max(n, 1), 32));
    if (n > LEAF) {
        binvL = alloc_view<V>(p, sbld, (long)ceil_div(n, SB) * sbld);
        binvU = alloc_view<V>(p, sbld, (long)ceil_div(n, SB) * sbld);
        tmp_cols = std::max<long>(n, 256);
        tmp = alloc_view<V>(p, sbld, tmp_cols);
    }
    la_cols = 0;
    if (look_ahead && n >= LA_MIN_N) {
        la_cols = round_up(n / 2, 256);
        for (int d = 0; d < NLA; ++d) la_tmp[d] = alloc_view<V>(p, sbld, la_cols);
    }
    refuted = (int *)take(256);
    wave_sync = (unsigned *)take(sizeof(unsigned) * (8 + 4 * NLA) * 256);
    perm = (int *)take(sizeof(int) * (size_t)nblk * PERM_STRIDE);
    cand_val = (T *)take(sizeof(T) * 2 * MAXG);
    cand_row = (int *)take(sizeof(int) * 2 * MAXG);
    cand_data = (E *)take(sizeof(E) * 2 * MAXG * IB);
    jrow = (E *)take(sizeof(E) * 2 * IB);
    counter = (unsigned *)take(256);
    slots = (unsigned long long *)take(sizeof(unsigned long long) * LL_WORDS);
    return (size_t)(p - (char *)base);
}
template <class V> size_t LuWork<V>::bytes(int n, bool look_ahead) {
    LuWork<V> tmp;
    return tmp.carve((void *)0, n, look_ahead);
}

// ------------------------------------------------------------------------------------------------- row interchanges
constexpr int SWP_CW = 16;  // columns per CTA
constexpr int SWP_NT = 256;

// Apply the net permutations of swap batches [b0, b1) in order to the columns [lo1,hi1) U [lo2,hi2) of A.
template <class V>
__global__ void __launch_bounds__(SWP_NT) laswp_kernel(V A, int lo1, int hi1, int lo2, int hi2, const int *perm, int b0, int b1) {
    typedef typename V::elem_t E;
    const int n1 = hi1 - lo1, ntot = n1 + (hi2 - lo2);
    const int tid = threadIdx.x;
    const int q = tid & (2 * IB - 1);          // pair slot 0..63
    const int cl = tid >> 6;                   // 0..3; columns cl, cl+4, cl+8, cl+12 of this CTA's group
    long col[SWP_CW / 4];
    bool cok[SWP_CW / 4];
#pragma unroll
    for (int e = 0; e < SWP_CW / 4; ++e) {
        int v = blockIdx.x * SWP_CW + cl + 4 * e;
        cok[e] = v < ntot;
        col[e] = v < n1 ? lo1 + v : lo2 + (v - n1);
    }
    for (int b = b0; b < b1; ++b) {
        const int *pb = perm + (size_t)b * PERM_STRIDE;
        const int cnt = pb[0];
        if (cnt == 0) continue;  // uniform across the CTA
        E val[SWP_CW / 4];
        int dst = 0;
        if (q < cnt) {
            dst = pb[1 + q];
            const int src = pb[1 + 2 * IB + q];
#pragma unroll
            for (int e = 0; e < SWP_CW / 4; ++e)
                if (cok[e]) val[e] = A.get(src, col[e]);
        }
        __syncthreads();
        if (q < cnt) {
#pragma unroll
            for (int e = 0; e < SWP_CW / 4; ++e)
                if (cok[e]) A.set(dst, col[e], val[e]);
        }
        __syncthreads();
    }
}

template <class V> static int laswp(cudaStream_t st, V A, int lo1, int hi1, int lo2, int hi2, const int *perm, int b0, int b1) {
    int ntot = (hi1 - lo1) + (hi2 - lo2);
    if (ntot <= 0 || b1 <= b0) return 0;
    ProfCat pc(PROF_LASWP);
    const bool prof = prof_enabled();
    if (prof) prof_begin(st, 0.0);
    laswp_kernel<V><<<ceil_div(ntot, SWP_CW), SWP_NT, 0, st>>>(A, lo1, hi1, lo2, hi2, perm, b0, b1);
    if (prof) prof_end(st);
    HP_LAUNCHED();
    return 0;
}

// ------------------------------------------------------------------------------------------------- inverse doubling
// Inverse of the w x w diagonal block at (c0,c0) from the inverses of its two diagonal sub-blocks a = [0,h), b = [h,w):
//     inv(L) = [ inv(La)                 0      ]      inv(U) = [ inv(Ua)   -inv(Ua) Uab inv(Ub) ]
//              [ -inv(Lb) Lba inv(La)   inv(Lb) ]               [   0              inv(Ub)       ]
// blockIdx.y = 0: L, 1: U.  Each CTA produces INV_RS rows of the w x w result; the off-diagonal part is
// out[I,:] = -(XL[I,:] * M) * XR with XL p x p, M p x q (the factor block), XR q x q.
constexpr int INV_RS = 16, INV_NT = 256;

template <class V>
__global__ void __launch_bounds__(INV_NT) inv_double_kernel(V A, int h, int w, V La, V Lb, V Lout, V Ua, V Ub, V Uout) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    extern __shared__ __align__(16) unsigned char smraw[];
    const bool isU = blockIdx.y == 1;
    const int i0 = blockIdx.x * INV_RS;            // first row of this strip inside the w x w block
    const int nr = min(INV_RS, w - i0);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const V Xa = isU ? Ua : La, Xb = isU ? Ub : Lb, O = isU ? Uout : Lout;
    const int hb = w - h;
    const bool top = i0 < h;
    pdl_wait();
    pdl_trigger();
    // rows that are plain copies / zeros
    if (top != isU) {
        // L top rows: [inv(La) | 0];  U bottom rows: [0 | inv(Ub)]
        for (int idx = tid; idx < nr * w; idx += INV_NT) {
            const int r = idx % nr, c = idx / nr;
            E v = mk((T)0, (T)0);
            if (!isU) { if (c < h) v = Xa.get(i0 + r, c); }
            else      { if (c >= h) v = Xb.get(i0 + r - h, c - h); }
            O.set(i0 + r, c, v);
        }
        return;
    }
    // L bottom rows: [-(inv(Lb)[I,:] Lba) inv(La) | inv(Lb)[I,:]];  U top rows: [inv(Ua)[I,:] | -(inv(Ua)[I,:] Uab) inv(Ub)]
    const int p = isU ? h : hb, q = isU ? hb : h;
    const V XL = isU ? Xa : Xb, XR = isU ? Xb : Xa;
    const V M = isU ? A.sub(0, h) : A.sub(h, 0);   // p x q factor block
    const int li0 = isU ? i0 : i0 - h;             // row offset inside XL
    const int ocol = isU ? h : 0;                  // column offset of the product inside the output
    constexpr int HL = LEAF / 2;                   // p, q <= HL
    E *xs = reinterpret_cast<E *>(smraw);          // [p][INV_RS]: XL[I, k] at xs[k*INV_RS + r]
    E *ts = xs + (size_t)HL * INV_RS;              // [q][INV_RS]: T[r, j] at ts[j*INV_RS + r]
    E *ms = ts + (size_t)HL * INV_RS;              // [q][p]: M[k, j] at ms[j*p + k]   (column-major, as in memory)
    E *xr = ms + (size_t)HL * HL;                  // [q][q]: XR[j, c] at xr[c*q + j]
    for (int idx = tid; idx < INV_RS * p; idx += INV_NT) {
        const int r = idx % INV_RS, k = idx / INV_RS;
        xs[idx] = r < nr ? XL.get(li0 + r, k) : mk((T)0, (T)0);
    }
    for (int idx = tid; idx < p * q; idx += INV_NT) ms[idx] = M.get(idx % p, idx / p);
    for (int idx = tid; idx < q * q; idx += INV_NT) xr[idx] = XR.get(idx % q, idx / q);
    // the diagonal-block copy of this strip
    for (int idx = tid; idx < nr * p; idx += INV_NT) {
        const int r = idx % nr, c = idx / nr;
        O.set(i0 + r, (isU ? 0 : h) + c, XL.get(li0 + r, c));
    }
    __syncthreads();
    // thread = row r of the strip x columns jg, jg + 16, jg + 32, jg + 48
    const int r = tid % INV_RS, jg = tid / INV_RS;
    constexpr int NJ = HL / (INV_NT / INV_RS);
    {   // phase 1: T = XL[I,:] * M
        E acc[NJ];
#pragma unroll
        for (int t = 0; t < NJ; ++t) acc[t] = mk((T)0, (T)0);
        for (int k = 0; k < p; ++k) {
            const E x = xs[k * INV_RS + r];
            const E nx = mk(-x.x, -x.y);
#pragma unroll
            for (int t = 0; t < NJ; ++t) {
                const int j = jg + (INV_NT / INV_RS) * t;
                if (j < q) acc[t] = cfnma(acc[t], nx, ms[j * p + k]);
            }
        }
#pragma unroll
        for (int t = 0; t < NJ; ++t) {
            const int j = jg + (INV_NT / INV_RS) * t;
            if (j < q) ts[j * INV_RS + r] = acc[t];
        }
    }
    __syncthreads();
    {   // phase 2: out = -T * XR
        E acc[NJ];
#pragma unroll
        for (int t = 0; t < NJ; ++t) acc[t] = mk((T)0, (T)0);
        for (int j = 0; j < q; ++j) {
            const E tv = ts[j * INV_RS + r];
#pragma unroll
            for (int t = 0; t < NJ; ++t) {
                const int c = jg + (INV_NT / INV_RS) * t;
                if (c < q) acc[t] = cfnma(acc[t], tv, xr[c * q + j]);
            }
        }
#pragma unroll
        for (int t = 0; t < NJ; ++t) {
            const int c = jg + (INV_NT / INV_RS) * t;
            if (c < q && r < nr) O.set(i0 + r, ocol + c, acc[t]);
        }
    }
}

// ------------------------------------------------------------------------------------------------- host recursion
// Column split of a node of width w: below LEAF the tree is binary on power-of-two multiples of IB, so that every left
// child is a full block of its size class (its inverse is kept, see LuWork); above, splits fall on multiples of LEAF, and
// above SB on multiples of SB, so that every SB-aligned block is a node of the recursion (its full inverse is kept too).
template <class V> static inline int split(int w) {
    constexpr int SB = SolveBlock<V>::value;
    if (w > SB) return (int)round_up((w + 1) / 2, SB);
    if (w > LEAF) return (int)round_up((w + 1) / 2, LEAF);
    int h = IB;
    while (2 * h < w) h *= 2;
    return h;
}
static inline int level_of(int w) {
    int lev = 0;
    while ((IB << lev) < w) ++lev;
    return lev;
}
// inverse of the (unit-lower | upper) triangle of the diagonal block of size s (<= LEAF) at offset d0 (a multiple of its
// size class)
template <class V> static V dinv_of(const V *tab, int d0, int s) {
    const int lev = level_of(s);
    const long sz = (long)IB << lev;
    return tab[lev].sub(0, (long)(d0 / sz) * sz);
}

template <class V> static int inv_double(cudaStream_t st, V A, int c0, int h, int w, LuWork<V> &wk) {
    typedef typename V::elem_t E;
    V La = dinv_of(wk.dinvL, c0, h), Lb = dinv_of(wk.dinvL, c0 + h, w - h), Lo = dinv_of(wk.dinvL, c0, w);
    V Ua = dinv_of(wk.dinvU, c0, h), Ub = dinv_of(wk.dinvU, c0 + h, w - h), Uo = dinv_of(wk.dinvU, c0, w);
    constexpr int HL = LEAF / 2;  // p, q <= LEAF/2
    const size_t smem = (2 * (size_t)HL * INV_RS + 2 * (size_t)HL * HL) * sizeof(E);
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, inv_double_kernel<V>, smem));
    ProfCat pc(PROF_OTHER);
    const bool prof = prof_enabled();
    if (prof) prof_begin(st, 0.0);
    HP_CUDA(launch_pdl(inv_double_kernel<V>, dim3(ceil_div(w, INV_RS), 2), dim3(INV_NT), smem, st, A.sub(c0, c0), h, w, La, Lb, Lo,
                       Ua, Ub, Uo));
    if (prof) prof_end(st);
    HP_LAUNCHED();
    return 0;
}

template <class V> static int panel(cudaStream_t st, int n, V A, int c0, int w, int *ipiv, int *info_dev, LuWork<V> &wk) {
    const int m = n - c0;
    const int blk = c0 / IB;
    V dl = wk.dinvL[0].sub(0, (long)blk * IB), du = wk.dinvU[0].sub(0, (long)blk * IB);
    int *perm = wk.perm + (size_t)blk * PERM_STRIDE;
    {
        ProfCat pc(PROF_PANEL);
        const bool prof = prof_enabled();
        if (prof) prof_begin(st, 0.0);
        const int rc = panel_launch<V>(st, A.sub(c0, c0), m, w, c0, ipiv, info_dev, wk, dl, du, perm);
        if (prof) prof_end(st);
        HP_TRY(rc);
    }
    HP_LAUNCHED();
    // this batch's interchanges on every other column of the matrix
    return laswp(st, A, 0, c0, c0 + w, n, wk.perm, blk, blk + 1);
}


// ---- helpers of the SB-block ("big leaf") level -------------------------------------------------------------------------
template <class V> __global__ void __launch_bounds__(256) set_identity_kernel(V X, int s) {
    typedef typename V::real_t T;
    const long idx = (long)blockIdx.x * 256 + threadIdx.x;
    if (idx >= (long)s * s) return;
    const int i = (int)(idx % s), j = (int)(idx / s);
    X.set(i, j, mk((T)(i == j ? 1 : 0), (T)0));
}
template <class V> __global__ void __launch_bounds__(256) copy_block_kernel(V Src, V Dst, int rows, long cols) {
    const long idx = (long)blockIdx.x * 256 + threadIdx.x;
    pdl_wait();
    pdl_trigger();
    if (idx >= (long)rows * cols) return;
    const int i = (int)(idx % rows);
    const long j = idx / rows;
    Dst.set(i, j, Src.get(i, j));
}
// zero the LEAF x LEAF diagonal blocks of the s x s matrix X
template <class V> __global__ void __launch_bounds__(256) strip_diag_kernel(V X, int s) {
    typedef typename V::real_t T;
    const long idx = (long)blockIdx.x * 256 + threadIdx.x;
    if (idx >= (long)s * LEAF) return;
    const int i = (int)(idx % s), jj = (int)(idx / s);  // jj: column inside the diagonal block of row i
    const int j = (i / LEAF) * LEAF + jj;
    if (j < s) X.set(i, j, mk((T)0, (T)0));
}
template <class V> static int copy_block(cudaStream_t st, V Src, V Dst, int rows, long cols) {
    if (rows <= 0 || cols <= 0) return 0;
    HP_CUDA(launch_pdl(copy_block_kernel<V>, dim3(ceil_div((long)rows * cols, 256)), dim3(256), 0, st, Src, Dst, rows, cols));
    HP_LAUNCHED();
    return 0;
}
// does the SB-aligned block starting at d0 have a kept full inverse, and is [d0, d0 + s) exactly that block?
template <class V> static inline bool is_big_block(int n, int d0, int s) {
    constexpr int SB = SolveBlock<V>::value;
    return d0 % SB == 0 && s > LEAF && s == std::min(SB, n - d0);
}
template <class V> static V binv_of(const V &tab, long sbld, int d0) { return tab.sub(0, (long)(d0 / SolveBlock<V>::value) * sbld); }

// the (batched) 3xTF32 product with the LEAF-diagonal blocks of an SB block, complex64 type only
static int diag_blocks_product(cudaStream_t, const ZView *, int, int, ZView, int, ZView) { return 0; }
static int diag_blocks_product(cudaStream_t st, const CView *dtab, int d0, int s, CView B, int ncols, CView T) {
    const int nfull = s / LEAF, rag = s - nfull * LEAF;
    const CView D = dtab[NLEV - 1].sub(0, (long)(d0 / LEAF) * LEAF);  // blocks contiguous: stride LEAF*LEAF
    if (nfull > 0)
        HP_TRY(cgemm3_batched(st, LEAF, ncols, LEAF, 1.0, D, (long)LEAF * LEAF, B, LEAF, 0.0, T, LEAF, nfull));
    if (rag > 0)
        HP_TRY(cgemm3(st, rag, ncols, rag, 1.0, dinv_of(dtab, d0 + nfull * LEAF, rag), B.sub(nfull * LEAF, 0), 0.0,
                      T.sub(nfull * LEAF, 0)));
    return 0;
}
// product inside the factorisation / the solves: FP32-class arithmetic when the workspace asks for it (complex64 only)
static int lu_gemm(const LuWork<ZView> &, cudaStream_t st, int m, int n, int k, double alpha, ZView A, ZView B, double beta, ZView C) {
    return gemm(st, m, n, k, alpha, A, B, beta, C);
}
static int lu_gemm(const LuWork<CView> &wk, cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta,
                   CView C) {
    if (wk.accurate) return cgemm3_any(st, m, n, k, alpha, A, B, beta, C);
    LuWork<CView> &w = const_cast<LuWork<CView> &>(wk);
    unsigned *slot = w.wave_sync ? w.wave_sync + 256 * (w.wave_base + (w.wave_next++ & w.wave_mask)) : nullptr;
    return cgemm_ws(st, m, n, k, alpha, A, B, beta, C, slot);
}
template <class V> struct IsPlanar { static constexpr bool value = false; };
template <> struct IsPlanar<CView> { static constexpr bool value = true; };

// B <- inv * B for an SB block: out of place into the scratch, then copied back.  acc (complex64 solves): the kept inverse
// has its LEAF-diagonal blocks zeroed; those are applied from the dinv table with the 3xTF32 kernel.
template <class V>
static int big_leaf(cudaStream_t st, const V &binv, const V *dtab, int d0, int s, V B, int ncols, LuWork<V> &wk, bool acc) {
    const long cap = wk.tmp_cols;
    for (long c = 0; c < ncols; c += cap) {
        const int nc = (int)std::min<long>(cap, ncols - c);
        V Bc = B.sub(0, c), T = wk.tmp;
        if (acc && IsPlanar<V>::value) {
            HP_TRY(diag_blocks_product(st, dtab, d0, s, Bc, nc, T));
            HP_TRY(lu_gemm(wk, st, s, nc, s, 1.0, binv_of(binv, wk.sbld, d0), Bc, 1.0, T));
        } else {
            HP_TRY(lu_gemm(wk, st, s, nc, s, 1.0, binv_of(binv, wk.sbld, d0), Bc, 0.0, T));
        }
        HP_TRY(copy_block(st, T, Bc, s, nc));
    }
    return 0;
}

// Leaf product of the triangular solves (inverted diagonal block times the right-hand sides): acc = FP32-class accuracy
// for the complex64 type (3xTF32).  The diagonal blocks are O(1) (their rounding to 10 mantissa bits would cap the solve
// at ~1e-3); the off-diagonal updates B2 -= L21 X1 stay single-pass like the trailing update of the factorisation, their
// error being 2^-11 |L21| |X1| with |L21| the (small) coupling entries.
static int gemm_sel(bool, cudaStream_t st, int m, int n, int k, double alpha, ZView A, ZView B, double beta, ZView C) {
    return gemm(st, m, n, k, alpha, A, B, beta, C);
}
static int gemm_sel(bool acc, cudaStream_t st, int m, int n, int k, double alpha, CView A, CView B, double beta, CView C) {
    return acc ? cgemm3(st, m, n, k, alpha, A, B, beta, C) : gemm(st, m, n, k, alpha, A, B, beta, C);
}

// LEAF product  B <- dinv * B  (s <= LEAF).  The complex128 type goes out of place through the scratch when the shape suits
// the 3M kernel (it cannot run in place: several M tiles per column strip) and copies back; everything else multiplies in
// place with the one-M-tile kernels.  Not while the kept block inverses are being built (use_big == false): that runs on
// the side stream, concurrently with leaf products of the main stream that own the scratch.  cfg 1: 53.4 -> 50.5 ms per step,
// cfg 3: 1318 -> 1306 ms.
static int leaf_product(bool acc, cudaStream_t st, int s, int ncols, ZView dinv, ZView B, LuWork<ZView> &wk) {
    if (wk.use_big && wk.tmp.p && s > 64 && ncols > 32 && ncols <= wk.tmp_cols) {
        HP_TRY(gemm(st, s, ncols, s, 1.0, dinv, B, 0.0, wk.tmp));
        return copy_block(st, wk.tmp, B, s, ncols);
    }
    return gemm_sel(acc, st, s, ncols, s, 1.0, dinv, B, 0.0, B);
}
static int leaf_product(bool acc, cudaStream_t st, int s, int ncols, CView dinv, CView B, LuWork<CView> &wk) {
    return gemm_sel(acc || wk.accurate, st, s, ncols, s, 1.0, dinv, B, 0.0, B);
}

// B <- L^-1 B, L = unit lower triangle of the s x s diagonal block of A at (d0,d0); B is s x ncols.  d0 is a multiple of
// LEAF, or s <= LEAF is a full block of its size class (or the ragged last block).
template <class V> static int trsm_lower(cudaStream_t st, V A, int d0, int s, V B, int ncols, LuWork<V> &wk, bool acc = false) {
    if (s <= 0 || ncols <= 0) return 0;
    if (s <= LEAF) return leaf_product(acc, st, s, ncols, dinv_of(wk.dinvL, d0, s), B, wk);
    if (wk.use_big && (acc || IsPlanar<V>::value) && is_big_block<V>(wk.n, d0, s))
        return big_leaf(st, wk.binvL, wk.dinvL, d0, s, B, ncols, wk, acc);
    const int h = split<V>(s);
    HP_TRY(trsm_lower(st, A, d0, h, B, ncols, wk, acc));
    HP_TRY(lu_gemm(wk, st, s - h, ncols, h, -1.0, A.sub(d0 + h, d0), B, 1.0, B.sub(h, 0)));
    return trsm_lower(st, A, d0 + h, s - h, B.sub(h, 0), ncols, wk, acc);
}

// B <- U^-1 B, U = upper triangle (with diagonal) of the s x s diagonal block of A at (d0,d0)
template <class V> static int trsm_upper(cudaStream_t st, V A, int d0, int s, V B, int ncols, LuWork<V> &wk, bool acc = false) {
    if (s <= 0 || ncols <= 0) return 0;
    if (s <= LEAF) return leaf_product(acc, st, s, ncols, dinv_of(wk.dinvU, d0, s), B, wk);
    if (wk.use_big && (acc || IsPlanar<V>::value) && is_big_block<V>(wk.n, d0, s))
        return big_leaf(st, wk.binvU, wk.dinvU, d0, s, B, ncols, wk, acc);
    const int h = split<V>(s);
    HP_TRY(trsm_upper(st, A, d0 + h, s - h, B.sub(h, 0), ncols, wk, acc));
    HP_TRY(lu_gemm(wk, st, h, ncols, s - h, -1.0, A.sub(d0, d0 + h), B.sub(h, 0), 1.0, B));
    return trsm_upper(st, A, d0, h, B, ncols, wk, acc);
}

// Full inverses of the unit-lower and upper triangles of the SB block [c0, c0 + s): triangular solves on the identity with
// the LEAF-level recursion (the block's own big leaf does not exist yet).
// What the factorisation itself does not need (for complex128 both inverses: its U12 solves keep the LEAF-level recursion,
// whose GEMMs run at full FP64 rate; for complex64 the upper one) is built on a side stream, under the rest of the LU.
// Raw entries (no context): one side stream + event pair per device, created on first use under a lock.  Host threads that
// share a device share it; every use is bracketed by its own fork/join events, so sharing only serialises side work.
struct SideRes {
    cudaStream_t s = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr;
};
static SideRes *pooled_side() {
    static std::mutex mu;
    static SideRes pool[32];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 32) return nullptr;
    std::lock_guard<std::mutex> lk(mu);
    SideRes &r = pool[dev];
    if (!r.s) {
        if (cudaStreamCreateWithFlags(&r.s, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&r.fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&r.join, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            r = SideRes();
            return nullptr;
        }
    }
    return &r;
}
template <class V> static SideRes side_of(const LuWork<V> &wk) {
    SideRes r;
    if (wk.side) {
        r.s = wk.side;
        r.fork = wk.ev_fork;
        r.join = wk.ev_join;
    } else if (SideRes *p = pooled_side()) {
        r = *p;
    }
    return r;
}
// `to` waits for everything enqueued on `from` so far
static int stream_follow(cudaStream_t from, cudaStream_t to, cudaEvent_t e) {
    HP_CUDA(cudaEventRecord(e, from));
    HP_CUDA(cudaStreamWaitEvent(to, e, 0));
    return 0;
}

template <class V> static int build_binv(cudaStream_t st, V A, int c0, int s, LuWork<V> &wk) {
    ProfCat pc(PROF_OTHER);
    V XL = binv_of(wk.binvL, wk.sbld, c0), XU = binv_of(wk.binvU, wk.sbld, c0);
    const SideRes sr = side_of(wk);
    cudaStream_t sd = sr.s ? sr.s : st;
    if (sd != st) HP_TRY(stream_follow(st, sd, sr.fork));
    cudaStream_t stl = IsPlanar<V>::value ? st : sd;  // the complex64 LU uses the lower inverse right away
    set_identity_kernel<V><<<ceil_div((long)s * s, 256), 256, 0, stl>>>(XL, s);
    HP_LAUNCHED();
    set_identity_kernel<V><<<ceil_div((long)s * s, 256), 256, 0, sd>>>(XU, s);
    HP_LAUNCHED();
    const bool was = wk.use_big;
    wk.use_big = false;
    int rc = trsm_lower(stl, A, c0, s, XL, s, wk, false);
    if (rc == 0) rc = trsm_upper(sd, A, c0, s, XU, s, wk, false);
    wk.use_big = was;
    if (sd != st) wk.side_used = true;
    return rc;
}

// pending: an event the RIGHT part of this node (the columns right of its left child) has to wait for -- the parent's
// look-ahead update of exactly those columns, running on another stream.  depth: look-ahead streams 0 .. depth - 1 may have
// work in flight, so this node and its sub-tree fork on stream `depth` and deeper.
template <class V>
static int getrf_rec(cudaStream_t st, int n, V A, int c0, int c1, int *ipiv, int *info_dev, LuWork<V> &wk,
                     cudaEvent_t pending = nullptr, int depth = 0) {
    const int w = c1 - c0;
    if ((wk.speculate && w <= TW) || w <= IB) {
        if (pending) HP_CUDA(cudaStreamWaitEvent(st, pending, 0));  // (not reached: look-ahead needs a node to wait in)
        if (wk.speculate) {
            ProfCat pc(PROF_PANEL);
            return block_panel<V>(st, n, A, c0, w, ipiv, info_dev, wk, dinv_of(wk.dinvL, c0, w), dinv_of(wk.dinvU, c0, w));
        }
        return panel(st, n, A, c0, w, ipiv, info_dev, wk);
    }
    const int h = split<V>(w), mid = c0 + h;
    HP_TRY(getrf_rec(st, n, A, c0, mid, ipiv, info_dev, wk, nullptr, pending ? depth + 1 : depth));
    if (pending) HP_CUDA(cudaStreamWaitEvent(st, pending, 0));
    // the right child's own left child spans [mid, mid + hr): only those columns are needed next
    const int wr = c1 - mid;
    const bool right_is_node = !((wk.speculate && wr <= TW) || wr <= IB);
    const int hr = right_is_node ? split<V>(wr) : wr;
    const bool ahead = IsPlanar<V>::value && wk.speculate && lookahead_enabled() && w <= LA_MAX_W && depth < LuWork<V>::NLA && wk.la_stream[depth] != nullptr &&
                       wk.la_cols > 0 && right_is_node && wr - hr >= LA_MIN_COLS && wr - hr <= wk.la_cols && !prof_enabled();
    const int now = ahead ? hr : wr;
    {
        ProfCat pc(PROF_LU_TRSM);
        HP_TRY(trsm_lower(st, A, c0, h, A.sub(c0, mid), now, wk));
    }
    {
        ProfCat pc(PROF_LU_GEMM);
        HP_TRY(lu_gemm(wk, st, n - mid, now, h, -1.0, A.sub(mid, c0), A.sub(c0, mid), 1.0, A.sub(mid, mid)));
    }
    cudaEvent_t join = nullptr;
    if (ahead) {
        // the rest of the update, under the factorisation of [mid, mid + hr): its own scratch, its own wave-barrier slots
        cudaStream_t sl = wk.la_stream[depth];
        HP_TRY(stream_follow(st, sl, wk.la_fork[depth]));
        LuWork<V> ws = wk;
        ws.tmp = wk.la_tmp[depth];
        ws.tmp_cols = wk.la_cols;
        ws.wave_base = 8 + 4 * depth;
        ws.wave_mask = 3;
        ws.wave_next = 0;
        const int later = wr - hr;
        ScopedSmReserve reserve(LA_SM_RESERVE);
        HP_TRY(trsm_lower(sl, A, c0, h, A.sub(c0, mid + hr), later, ws));
        HP_TRY(lu_gemm(ws, sl, n - mid, later, h, -1.0, A.sub(mid, c0), A.sub(c0, mid + hr), 1.0, A.sub(mid, mid + hr)));
        join = wk.la_join[depth];
        HP_CUDA(cudaEventRecord(join, sl));
    }
    HP_TRY(getrf_rec(st, n, A, mid, c1, ipiv, info_dev, wk, join, depth));
    // the node's diagonal block is final: keep its inverse for the triangular solves further up / in getrs
    if (w <= LEAF) HP_TRY(inv_double(st, A, c0, h, w, wk));
    if (is_big_block<V>(n, c0, w)) HP_TRY(build_binv(st, A, c0, w, wk));
    return 0;
}

template <class V> int getrf(cudaStream_t st, int n, V A, int *ipiv, int *info_dev, LuWork<V> &wk) {
    if (n <= 0) return 0;
    HP_CUDA(cudaMemsetAsync(wk.counter, 0, sizeof(unsigned), st));
    HP_CUDA(cudaMemsetAsync(wk.slots, 0, sizeof(unsigned long long) * LL_WORDS, st));
    HP_CUDA(cudaMemsetAsync(wk.refuted, 0, sizeof(int), st));
    wk.bar_base = 0;
    wk.ep_base = 0;
    wk.use_big = true;
    wk.side_used = false;
    HP_TRY(getrf_rec(st, n, A, 0, n, ipiv, info_dev, wk));
    if (wk.side_used) {  // join: the kept inverses are complete
        const SideRes sr = side_of(wk);
        HP_TRY(stream_follow(sr.s, st, sr.join));
    }
    if (IsPlanar<V>::value && n > LEAF) {
        // the solves apply the LEAF-diagonal blocks of the kept inverses separately, with FP32-class products
        ProfCat pc(PROF_OTHER);
        constexpr int SB = SolveBlock<V>::value;
        for (int d0 = 0; d0 < n; d0 += SB) {
            const int sblk = std::min(SB, n - d0);
            if (sblk <= LEAF) continue;
            strip_diag_kernel<V><<<ceil_div((long)sblk * LEAF, 256), 256, 0, st>>>(binv_of(wk.binvL, wk.sbld, d0), sblk);
            HP_LAUNCHED();
            strip_diag_kernel<V><<<ceil_div((long)sblk * LEAF, 256), 256, 0, st>>>(binv_of(wk.binvU, wk.sbld, d0), sblk);
            HP_LAUNCHED();
        }
    }
    return 0;
}

template <class V> int getrs(cudaStream_t st, int n, int nrhs, V A, V B, LuWork<V> &wk) {
    if (n <= 0 || nrhs <= 0) return 0;
    ProfCat pc(PROF_SOLVE);
    wk.use_big = true;
    // a factorisation with verified diagonal pivots has no interchanges (all swap batches are empty; a refuted one is never
    // solved with: the caller refactors with pivoting)
    if (!wk.speculate) HP_TRY(laswp(st, B, 0, nrhs, 0, 0, wk.perm, 0, wk.nblk));
    // the right-hand sides and the solution are O(1): FP32-class diagonal-block products (3xTF32 for the complex64 type)
    HP_TRY(trsm_lower(st, A, 0, n, B, nrhs, wk, true));
    return trsm_upper(st, A, 0, n, B, nrhs, wk, true);
}

template struct LuWork<CView>;
template int getrf<CView>(cudaStream_t, int, CView, int *, int *, LuWork<CView> &);
template int getrs<CView>(cudaStream_t, int, int, CView, CView, LuWork<CView> &);
template struct LuWork<ZView>;
template int getrf<ZView>(cudaStream_t, int, ZView, int *, int *, LuWork<ZView> &);
template int getrs<ZView>(cudaStream_t, int, int, ZView, ZView, LuWork<ZView> &);

}  // namespace hp
