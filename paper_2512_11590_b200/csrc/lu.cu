// lu.cu -- recursive blocked LU with partial pivoting, M = P L U (Eq. 5), and the triangular
// solves for the nch right-hand sides (PAPER.md:127 "forward and backward substitution"; :137 step 3).
//
// Structure:
//   getrf_rec(c0,c1): width <= IB -> panel kernel; else factor the left half, U12 <- L11^-1 A12 (recursive TRSM whose
//   leaves multiply by inverted IB x IB diagonal blocks), A22 <- A22 - L21 U12 (tensor-core GEMM), factor the right
//   half.  All O(N^3) work is GEMM with K up to N/2, so the trailing update is compute- not HBM-bound.
//   Panel: one cooperative kernel, one CTA per SM, each CTA keeps its slice of panel rows in shared memory for all IB
//   columns; per column one grid barrier: every CTA publishes its local pivot candidate ROW, all CTAs pick the same
//   winner and read its row, swap and rank-1 update locally.  The multipliers are scaled at write-back.
//   Row interchanges: right after each panel, its IB swaps are folded into one net permutation of <= 2 IB rows and
//   applied to ALL other columns of the matrix by a gather/scatter kernel (independent loads, no swap chain).
#include "lu.cuh"

#include <algorithm>

#include <cooperative_groups.h>

namespace hp {

constexpr int PANEL_NT = 256;
constexpr int PANEL_MINROWS = 128;
// exchange buffer of the register-resident panel kernel (layout: see "panel kernel, v2" below), in 8-byte words
constexpr int LL_SLOT_WORDS = 2;            // { epoch16 | 48 payload bits } x 2 = |candidate| (64 bits) + row (32 bits)
constexpr int LL_ROW_WORDS = IB * 4;        // room for IB double2 elements
constexpr size_t LL_SLOTS = 2 * (size_t)MAXG * MAXG * LL_SLOT_WORDS;     // words: one mailbox of MAXG slots per CTA and parity
constexpr size_t LL_ROWS = 2 * (size_t)(MAXG + 1) * LL_ROW_WORDS;        // words; row index MAXG = "row j"
constexpr size_t LL_WORDS = LL_SLOTS + LL_ROWS;

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

template <class V> size_t LuWork<V>::carve(void *base, int n_) {
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
    sbld = std::min<long>(SB, round_up(std::max(n, 1), 32));
    if (n > LEAF) {
        binvL = alloc_view<V>(p, sbld, (long)ceil_div(n, SB) * sbld);
        binvU = alloc_view<V>(p, sbld, (long)ceil_div(n, SB) * sbld);
        tmp = alloc_view<V>(p, sbld, std::max<long>(n, 256));
    }
    perm = (int *)take(sizeof(int) * (size_t)nblk * PERM_STRIDE);
    cand_val = (T *)take(sizeof(T) * 2 * MAXG);
    cand_row = (int *)take(sizeof(int) * 2 * MAXG);
    cand_data = (E *)take(sizeof(E) * 2 * MAXG * IB);
    jrow = (E *)take(sizeof(E) * 2 * IB);
    counter = (unsigned *)take(256);
    slots = (unsigned long long *)take(sizeof(unsigned long long) * LL_WORDS);
    return (size_t)(p - (char *)base);
}
template <class V> size_t LuWork<V>::bytes(int n) {
    LuWork<V> tmp;
    return tmp.carve((void *)0, n);
}

// ------------------------------------------------------------------------------------------------- panel kernel
__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// all CTAs of the (cooperatively launched, hence co-resident) grid arrive; counter is monotone, target = base + G*k
__device__ __forceinline__ void grid_barrier(unsigned *counter, unsigned target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(counter, 1u);
        while ((int)(ld_acquire_u32(counter) - target) < 0) {
        }
        __threadfence();
    }
    __syncthreads();
}

template <class T> __device__ __forceinline__ bool better(T v, int i, T bv, int bi) {
    // larger modulus wins; ties go to the smaller row index (first maximum, LAPACK's izamax)
    return (v > bv) || (v == bv && i >= 0 && (bi < 0 || i < bi));
}

template <class E> __device__ __forceinline__ E ldcg_e(const E *p);
template <> __device__ __forceinline__ double2 ldcg_e<double2>(const double2 *p) { return __ldcg(p); }
template <> __device__ __forceinline__ float2 ldcg_e<float2>(const float2 *p) { return __ldcg(p); }

// Net permutation of one swap batch: content of every touched row after the jb interchanges piv[] (panel-relative rows),
// written as (count, destination rows, source rows) with absolute row numbers.  One warp.
__device__ void net_permutation(const int *piv, int jb, int j0, int *perm, int lane) {
    // net permutation: content of every touched row after the jb interchanges (rows are panel-relative here)
    __shared__ int top[IB], orow[IB], ocont[IB];
    __shared__ int nout;
    if (lane == 0) nout = 0;
    for (int k = lane; k < jb; k += 32) top[k] = k;
    __syncwarp();
    for (int k = 0; k < jb; ++k) {
        const int pk = piv[k];
        if (pk == k) continue;
        if (pk < jb) {
            if (lane == 0) { int t = top[k]; top[k] = top[pk]; top[pk] = t; }
        } else {
            const int no = nout;
            int found = -1;
            if (lane < no && orow[lane] == pk) found = lane;
            unsigned bal = __ballot_sync(0xffffffffu, found >= 0);
            int idx = bal ? (__ffs(bal) - 1) : no;
            if (lane == 0) {
                if (!bal) { orow[idx] = pk; ocont[idx] = pk; nout = no + 1; }
                int t = top[k]; top[k] = ocont[idx]; ocont[idx] = t;
            }
        }
        __syncwarp();
    }
    if (lane == 0) {
        int cnt = 0;
        for (int k = 0; k < jb; ++k)
            if (top[k] != k) { perm[1 + cnt] = j0 + k; perm[1 + 2 * IB + cnt] = j0 + top[k]; ++cnt; }
        for (int q = 0; q < nout; ++q)
            if (ocont[q] != orow[q]) { perm[1 + cnt] = j0 + orow[q]; perm[1 + 2 * IB + cnt] = j0 + ocont[q]; ++cnt; }
        perm[0] = cnt;
    }
}

template <class V>
__global__ void __launch_bounds__(PANEL_NT, 1)
    panel_lu_kernel(V A, int m, int jb, int j0, int rpc, int *ipiv, int *info, typename V::real_t *cand_val,
                    int *cand_row, typename V::elem_t *cand_data, typename V::elem_t *jrow_g, unsigned *counter,
                    unsigned bar_base, V dinvL, V dinvU, int *perm) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    extern __shared__ __align__(16) unsigned char smraw[];
    E *chunk = reinterpret_cast<E *>(smraw);          // [IB][rpc], column-major slice of the panel
    E *inv_s = chunk + (size_t)IB * rpc;              // [2][IB][IB] scratch for the diagonal-block inverses (CTA 0)
    __shared__ E prow[IB], jr[IB], invp[IB];
    __shared__ int piv[IB];
    __shared__ T red_val[PANEL_NT / 32];
    __shared__ int red_idx[PANEL_NT / 32];
    __shared__ T s_bval;
    __shared__ int s_bli, s_win, s_p;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x, G = gridDim.x;
    const int row0 = cta * rpc;
    const int nloc = max(0, min(rpc, m - row0));

    for (int idx = tid; idx < jb * nloc; idx += PANEL_NT) {
        int c = idx / nloc, li = idx - c * nloc;
        chunk[c * rpc + li] = A.get(row0 + li, c);
    }
    __syncthreads();

    T myval = (T)-1;
    int myli = -1;
    for (int li = tid; li < nloc; li += PANEL_NT) {
        T v = cabs1(chunk[li]);
        if (v > myval) { myval = v; myli = li; }
    }

    for (int j = 0; j < jb; ++j) {
        const int par = j & 1;
        // ---- local arg-max of column j over this CTA's rows (global panel row >= j)
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            T ov = __shfl_down_sync(0xffffffffu, myval, off);
            int oi = __shfl_down_sync(0xffffffffu, myli, off);
            if (better(ov, oi, myval, myli)) { myval = ov; myli = oi; }
        }
        if (lane == 0) { red_val[warp] = myval; red_idx[warp] = myli; }
        __syncthreads();
        if (warp == 0) {
            T v = lane < PANEL_NT / 32 ? red_val[lane] : (T)-1;
            int i = lane < PANEL_NT / 32 ? red_idx[lane] : -1;
#pragma unroll
            for (int off = 4; off > 0; off >>= 1) {
                T ov = __shfl_down_sync(0xffffffffu, v, off);
                int oi = __shfl_down_sync(0xffffffffu, i, off);
                if (better(ov, oi, v, i)) { v = ov; i = oi; }
            }
            if (lane == 0) { s_bval = v; s_bli = i; }
        }
        __syncthreads();
        // ---- publish the candidate row (and row j, for the swap) and meet the other CTAs
        {
            const int bli = s_bli;
            if (tid < jb && bli >= 0) cand_data[(size_t)(par * MAXG + cta) * IB + tid] = chunk[tid * rpc + bli];
            if (tid == 0) {
                cand_val[par * MAXG + cta] = bli >= 0 ? s_bval : (T)-1;
                cand_row[par * MAXG + cta] = row0 + bli;
            }
            if (j >= row0 && j < row0 + nloc && tid >= 32 && tid < 32 + jb)
                jrow_g[par * IB + tid - 32] = chunk[(tid - 32) * rpc + j - row0];
        }
        grid_barrier(counter, bar_base + (unsigned)G * (unsigned)(j + 1));
        // ---- every CTA picks the same winner
        if (warp == 0) {
            T bv = (T)-1;
            int br = -1, bg = -1;
            for (int g = lane; g < G; g += 32) {
                T v = __ldcg(&cand_val[par * MAXG + g]);
                int rr = __ldcg(&cand_row[par * MAXG + g]);
                if (v >= (T)0 && better(v, rr, bv, br)) { bv = v; br = rr; bg = g; }
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                T ov = __shfl_down_sync(0xffffffffu, bv, off);
                int orr = __shfl_down_sync(0xffffffffu, br, off);
                int og = __shfl_down_sync(0xffffffffu, bg, off);
                if (og >= 0 && better(ov, orr, bv, br)) { bv = ov; br = orr; bg = og; }
            }
            if (lane == 0) { s_win = bg; s_p = bg >= 0 ? br : j; }
        }
        __syncthreads();
        const int p = s_p, win = s_win;
        const bool ownp = (p >= row0 && p < row0 + nloc), ownj = (j >= row0 && j < row0 + nloc);
        if (tid < jb) prow[tid] = win >= 0 ? ldcg_e(&cand_data[(size_t)(par * MAXG + win) * IB + tid]) : mk((T)0, (T)0);
        if (ownp && p != j && tid >= 32 && tid < 32 + jb) jr[tid - 32] = ldcg_e(&jrow_g[par * IB + tid - 32]);
        if (tid == 0) {
            piv[j] = p;
            if (cta == 0) ipiv[j0 + j] = j0 + p + 1;
        }
        __syncthreads();
        if (tid < jb) {
            if (ownp && p != j) chunk[tid * rpc + p - row0] = jr[tid];
            if (ownj) chunk[tid * rpc + j - row0] = prow[tid];
        }
        const E pv = prow[j];
        const bool sing = (pv.x == (T)0 && pv.y == (T)0);
        const E ip = sing ? mk((T)0, (T)0) : crecip(pv);
        if (tid == 0) {
            invp[j] = ip;
            if (sing && cta == 0) atomicCAS(info, 0, j0 + j + 1);
        }
        __syncthreads();
        // ---- rank-1 update of the local rows below the diagonal, fused with the next column's arg-max
        myval = (T)-1;
        myli = -1;
        if (!sing || j + 1 < jb) {
            for (int li = tid; li < nloc; li += PANEL_NT) {
                if (row0 + li > j) {
                    if (!sing) {
                        const E l = cmul(chunk[j * rpc + li], ip);
                        for (int c = j + 1; c < jb; ++c) chunk[c * rpc + li] = cfnma(chunk[c * rpc + li], l, prow[c]);
                    }
                    if (j + 1 < jb) {
                        T v = cabs1(chunk[(j + 1) * rpc + li]);
                        if (v > myval) { myval = v; myli = li; }
                    }
                }
            }
        }
    }
    __syncthreads();

    // ---- write back; multipliers are scaled by 1/pivot here
    for (int idx = tid; idx < jb * nloc; idx += PANEL_NT) {
        int c = idx / nloc, li = idx - c * nloc;
        E v = chunk[c * rpc + li];
        if (row0 + li > c) v = cmul(v, invp[c]);
        A.set(row0 + li, c, v);
    }

    if (cta != 0) return;
    // ---- CTA 0 owns the top jb x jb block: inverses of its unit-lower and upper triangles (leaves of the TRSM
    //      recursion), and the net row permutation of this swap batch.
    E *xl = inv_s, *xu = inv_s + IB * IB;  // column-major jb x jb, ld = IB
    if (tid < jb) {
        const int cc = tid;  // column cc of inv(L): forward substitution on e_cc
        for (int i = 0; i < jb; ++i) xl[cc * IB + i] = mk((T)(i == cc ? 1 : 0), (T)0);
        for (int i = cc + 1; i < jb; ++i) {
            E s = mk((T)0, (T)0);
            for (int k = cc; k < i; ++k) s = cadd(s, cmul(cmul(chunk[k * rpc + i], invp[k]), xl[cc * IB + k]));
            xl[cc * IB + i] = mk(-s.x, -s.y);
        }
        for (int i = 0; i < jb; ++i) dinvL.set(i, cc, xl[cc * IB + i]);
    } else if (tid >= 32 && tid < 32 + jb) {
        const int cc = tid - 32;  // column cc of inv(U): back substitution on e_cc
        for (int i = 0; i < jb; ++i) xu[cc * IB + i] = mk((T)0, (T)0);
        xu[cc * IB + cc] = invp[cc];
        for (int i = cc - 1; i >= 0; --i) {
            E s = mk((T)0, (T)0);
            for (int k = i + 1; k <= cc; ++k) s = cadd(s, cmul(chunk[k * rpc + i], xu[cc * IB + k]));
            E q = cmul(s, invp[i]);
            xu[cc * IB + i] = mk(-q.x, -q.y);
        }
        for (int i = 0; i < jb; ++i) dinvU.set(i, cc, xu[cc * IB + i]);
    } else if (warp == 2) {
        net_permutation(piv, jb, j0, perm, lane);
    }
}

// ------------------------------------------------------------------------------------------------- panel kernel, v2
// Register-resident variant: every thread owns RPT rows of the panel (all IB columns) in registers, so the rank-1 updates
// touch no memory, and the per-column exchange between the CTAs uses neither an atomic counter nor a memory fence.
// Everything that crosses CTAs travels as 8-byte words  { 32-bit payload | 32-bit epoch }  (the "LL" protocol of
// collective-communication libraries: an aligned 8-byte store is single-copy atomic, so a word whose epoch matches
// carries valid payload, whatever order the words arrive in).  Per column every CTA publishes
//   slot = { |pivot candidate| as a double, its row }  (two words of 16-bit epoch + 48 payload bits), pushed into the
//   mailbox of EVERY CTA (so that each CTA polls only its own lines: no L2 hot spot), and its candidate ROW;
// the owner of row j publishes row j (needed by the owner of the pivot row for the swap); one warp per CTA polls its
// mailbox -- "all G slots carry this column's epoch" is the barrier, the polled words already are the candidates --
// then reads the winner's row, spinning on its epochs.  All buffers are double-buffered by column parity: a CTA can be
// at most one column ahead of the slowest reader.

__device__ __forceinline__ void ld_relaxed_v2(const unsigned long long *p, unsigned long long &a, unsigned long long &b) {
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0,%1}, [%2];\n" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_relaxed_v2(unsigned long long *p, unsigned long long a, unsigned long long b) {
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1,%2};\n" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ unsigned long long ll_word(unsigned payload, unsigned flag) {
    return ((unsigned long long)flag << 32) | payload;
}
__device__ __forceinline__ bool ll_ok(unsigned long long w, unsigned flag) { return (unsigned)(w >> 32) == flag; }

// one matrix element <-> LL words at p (16-byte aligned)
__device__ __forceinline__ void ll_store(unsigned long long *p, float2 v, unsigned flag) {
    st_relaxed_v2(p, ll_word(__float_as_uint(v.x), flag), ll_word(__float_as_uint(v.y), flag));
}
__device__ __forceinline__ void ll_store(unsigned long long *p, double2 v, unsigned flag) {
    st_relaxed_v2(p, ll_word((unsigned)__double2loint(v.x), flag), ll_word((unsigned)__double2hiint(v.x), flag));
    st_relaxed_v2(p + 2, ll_word((unsigned)__double2loint(v.y), flag), ll_word((unsigned)__double2hiint(v.y), flag));
}
__device__ __forceinline__ bool ll_load(const unsigned long long *p, float2 &v, unsigned flag) {
    unsigned long long a, b;
    ld_relaxed_v2(p, a, b);
    v = make_float2(__uint_as_float((unsigned)a), __uint_as_float((unsigned)b));
    return ll_ok(a, flag) && ll_ok(b, flag);
}
__device__ __forceinline__ bool ll_load(const unsigned long long *p, double2 &v, unsigned flag) {
    unsigned long long a, b, c, d;
    ld_relaxed_v2(p, a, b);
    ld_relaxed_v2(p + 2, c, d);
    v = make_double2(__hiloint2double((int)(unsigned)b, (int)(unsigned)a), __hiloint2double((int)(unsigned)d, (int)(unsigned)c));
    return ll_ok(a, flag) && ll_ok(b, flag) && ll_ok(c, flag) && ll_ok(d, flag);
}
template <class E> struct LLWords;
template <> struct LLWords<float2> { static constexpr int n = 2; };
template <> struct LLWords<double2> { static constexpr int n = 4; };

// shared-memory loads through an explicit 32-bit shared address (one LDS, no generic-address arithmetic)
__device__ __forceinline__ void lds_e(unsigned addr, float2 &v) {
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];\n" : "=f"(v.x), "=f"(v.y) : "r"(addr));
}
__device__ __forceinline__ void lds_e(unsigned addr, double2 &v) {
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];\n" : "=d"(v.x), "=d"(v.y) : "r"(addr));
}

// 1/a by Smith's formula on the reciprocal intrinsics (two dependent reciprocals, no IEEE-division slow paths)
__device__ __forceinline__ float rcp_rn(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double rcp_rn(double x) { return __drcp_rn(x); }
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

// Warp-wide arg-max of (v, li): v >= 0 a modulus (or li < 0: no candidate); the largest v wins, ties go to the smallest
// li.  Integer redux.sync on the (order-preserving) bit patterns.  Result valid in every lane; li = -1 if none.
__device__ __forceinline__ void warp_argmax(float &v, int &li) {
    const unsigned b = li >= 0 ? __float_as_uint(v) : 0u;
    const unsigned mb = __reduce_max_sync(0xffffffffu, b);
    const int idx = __reduce_min_sync(0xffffffffu, (li >= 0 && b == mb) ? li : 0x7fffffff);
    v = __uint_as_float(mb);
    li = idx == 0x7fffffff ? -1 : idx;
}
__device__ __forceinline__ void warp_argmax(double &v, int &li) {
    const unsigned hi = li >= 0 ? (unsigned)__double2hiint(v) : 0u;
    const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
    const unsigned lo = (li >= 0 && hi == mh) ? (unsigned)__double2loint(v) : 0u;
    const unsigned ml = __reduce_max_sync(0xffffffffu, lo);
    const int idx = __reduce_min_sync(0xffffffffu, (li >= 0 && hi == mh && lo == ml) ? li : 0x7fffffff);
    v = __hiloint2double((int)mh, (int)ml);
    li = idx == 0x7fffffff ? -1 : idx;
}

// compile-time loop: f(integral_constant<int, I>) for I = B .. E-1 (keeps the register-resident panel statically indexed)
template <int I> struct IntC { static constexpr int value = I; };
template <int B, int E_, class F> __device__ __forceinline__ void static_for(F &&f) {
    if constexpr (B < E_) {
        f(IntC<B>{});
        static_for<B + 1, E_>(f);
    }
}

template <class V, int RPT, bool TIMING = false>
__global__ void __launch_bounds__(PANEL_NT, 1)
    panel_reg_kernel(V A, int m, int jb, int j0, int rpc, int *ipiv, int *info, unsigned long long *ll, unsigned ep_base,
                     V dinvL, V dinvU, int *perm, long long *dbg) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
    extern __shared__ __align__(16) unsigned char smraw[];
    E *topb = reinterpret_cast<E *>(smraw);  // [IB][IB] column-major copy of the panel's top block (CTA 0)
    E *inv_s = topb + IB * IB;               // [2][IB][IB] scratch for its triangular inverses (CTA 0)
    __shared__ __align__(16) E prow[IB + 4];
    __shared__ E jr[IB], invp[IB];
    __shared__ int piv[IB];
    __shared__ T red_val[PANEL_NT / 32];
    __shared__ int red_idx[PANEL_NT / 32];
    __shared__ int s_p;
    __shared__ E s_ip;
    constexpr int NW = LLWords<E>::n;
    constexpr int POLLW = PANEL_NT / 32 - 1;  // the warp that talks to the other CTAs: the one owning the fewest rows
    unsigned long long *ll_slots = ll, *ll_rows = ll + LL_SLOTS;
    const unsigned prow_s = (unsigned)__cvta_generic_to_shared(prow);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x, G = gridDim.x;
    const int row0 = cta * rpc;
    const int nloc = max(0, min(rpc, m - row0));

    long long tph[6] = {0, 0, 0, 0, 0, 0}, tlast = 0;  // TIMING: cycles of thread 0 per phase
    auto tick = [&](int ph) {
        if constexpr (TIMING) {
            const long long now = clock64();
            tph[ph] += now - tlast;
            tlast = now;
        }
    };
    if constexpr (TIMING) tlast = clock64();
    E a[RPT][IB];
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const int li = tid + r * PANEL_NT;
#pragma unroll
        for (int c = 0; c < IB; ++c) a[r][c] = (li < nloc && c < jb) ? A.get(row0 + li, c) : mk((T)0, (T)0);
    }
    tick(0);

    T myval = (T)-1;
    int myli = -1;
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const int li = tid + r * PANEL_NT;
        if (li < nloc) {
            const T v = cabs1(a[r][0]);
            if (v > myval) { myval = v; myli = li; }
        }
    }

    // Rolled loop over the columns (compact code: the fully unrolled form thrashes the instruction cache).  The register
    // window rotates left by one column per step, so the current column is always a[.][0], the still-active columns
    // are a[.][1 .. IB-1-j] and the finished ones follow; all indices stay compile-time.  After IB rotations the
    // window is back in natural order.  Candidate rows / row j travel in the same rotated frame on every CTA.
#pragma unroll 1
    for (int j = 0; j < IB; ++j) {
        if (j < jb) {  // uniform
            const int par = j & 1;
            const unsigned flag = ep_base + (unsigned)j + 1u;
            // ---- local arg-max of column j: redux.sync inside the warps, then every warp folds the per-warp results
            warp_argmax(myval, myli);
            if (lane == 0) { red_val[warp] = myval; red_idx[warp] = myli; }
            __syncthreads();
            T bval = lane < PANEL_NT / 32 ? red_val[lane] : (T)0;
            int bli = lane < PANEL_NT / 32 ? red_idx[lane] : -1;
            warp_argmax(bval, bli);
            tick(1);
            // ---- publish: the candidate's value and row (thread 0), the candidate row and row j (their owners)
            if (warp == POLLW) {
                // push this CTA's candidate into every CTA's mailbox (each CTA then polls only its own lines)
                const unsigned long long vb = bli >= 0 ? (unsigned long long)__double_as_longlong((double)bval) : 0ull;
                const unsigned long long ep = (unsigned long long)(flag & 0xffffu) << 48;
                const unsigned long long s0 = ep | (vb >> 16);
                const unsigned long long s1 = ep | ((vb & 0xffffull) << 32) | (bli >= 0 ? (unsigned)(row0 + bli) : 0xffffffffu);
                for (int g = lane; g < G; g += 32)
                    st_relaxed_v2(ll_slots + ((size_t)(g * 2 + par) * MAXG + cta) * LL_SLOT_WORDS, s0, s1);
            }
            {
                const int lj = j - row0;
#pragma unroll
                for (int r = 0; r < RPT; ++r) {
                    const int li = tid + r * PANEL_NT;
                    if (li == bli) {
                        unsigned long long *dst = ll_rows + (size_t)(par * (MAXG + 1) + cta) * LL_ROW_WORDS;
#pragma unroll
                        for (int c = 0; c < IB; ++c) ll_store(dst + c * NW, a[r][c], flag);
                    }
                    if (li == lj && lj < nloc) {
                        unsigned long long *dst = ll_rows + (size_t)(par * (MAXG + 1) + MAXG) * LL_ROW_WORDS;
#pragma unroll
                        for (int c = 0; c < IB; ++c) ll_store(dst + c * NW, a[r][c], flag);
                    }
                }
            }
            tick(2);
            // ---- all CTAs' candidates: poll until every slot carries this column's epoch, pick the same winner
            if (warp == POLLW) {
                constexpr int NS = (MAXG + 31) / 32;
                // each lane watches the slots g = lane + 32 q; only slots not yet seen with this epoch are re-read
                unsigned long long w0[NS], w1[NS];
                unsigned have = 0;
                const unsigned long long ep = (unsigned long long)(flag & 0xffffu);
#pragma unroll
                for (int q = 0; q < NS; ++q)
                    if (lane + 32 * q >= G) have |= 1u << q;
                do {
#pragma unroll
                    for (int q = 0; q < NS; ++q)
                        if (!(have >> q & 1u))
                            ld_relaxed_v2(ll_slots + ((size_t)(cta * 2 + par) * MAXG + lane + 32 * q) * LL_SLOT_WORDS, w0[q], w1[q]);
#pragma unroll
                    for (int q = 0; q < NS; ++q)
                        if (!(have >> q & 1u) && (w0[q] >> 48) == ep && (w1[q] >> 48) == ep) have |= 1u << q;
                } while (!__all_sync(0xffffffffu, have == (1u << NS) - 1u));
                tick(3);
                double bv = -1.0;
                int br = -1;
#pragma unroll
                for (int q = 0; q < NS; ++q) {
                    if (lane + 32 * q < G) {
                        const int rr = (int)(unsigned)w1[q];
                        const double v = __longlong_as_double((long long)(((w0[q] & 0xffffffffffffull) << 16) | ((w1[q] >> 32) & 0xffffull)));
                        if (rr >= 0 && better(v, rr, bv, br)) { bv = v; br = rr; }
                    }
                }
                warp_argmax(bv, br);  // largest modulus, smallest row on ties; br = -1: nobody has a candidate
                const int bg = br >= 0 ? br / rpc : -1;
                const int p = bg >= 0 ? br : j;
                const bool needj = (p != j && p >= row0 && p < row0 + nloc);
                E pe = mk((T)0, (T)0), je = mk((T)0, (T)0);
                {
                    const unsigned long long *srcp = ll_rows + (size_t)(par * (MAXG + 1) + max(bg, 0)) * LL_ROW_WORDS + lane * NW;
                    const unsigned long long *srcj = ll_rows + (size_t)(par * (MAXG + 1) + MAXG) * LL_ROW_WORDS + lane * NW;
                    bool okp = bg < 0, okj = !needj;
                    while (!(okp && okj)) {  // both loads in flight together
                        E tp, tj;
                        bool gp = false, gj = false;
                        if (!okp) gp = ll_load(srcp, tp, flag);
                        if (!okj) gj = ll_load(srcj, tj, flag);
                        if (gp) { pe = tp; okp = true; }
                        if (gj) { je = tj; okj = true; }
                    }
                }
                prow[lane] = pe;
                jr[lane] = je;
                if (lane == 0) {
                    const bool sing0 = (pe.x == (T)0 && pe.y == (T)0);
                    const E ip0 = sing0 ? mk((T)0, (T)0) : crecip_fast(pe);
                    s_ip = ip0;
                    invp[j] = ip0;
                    s_p = p;
                    piv[j] = p;
                    if (cta == 0) {
                        ipiv[j0 + j] = j0 + p + 1;
                        if (sing0) atomicCAS(info, 0, j0 + j + 1);
                    }
                }
            }
            __syncthreads();
            tick(4);
            const int p = s_p;
            const E ip = s_ip;
            const bool sing = (ip.x == (T)0 && ip.y == (T)0);
            // ---- interchange, multipliers, rank-1 update of the active window (all in registers), next arg-max
            myval = (T)-1;
            myli = -1;
            const int nact = IB - 1 - j;  // active columns after this one: window positions 1 .. nact
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const int li = tid + r * PANEL_NT;
                const int grow = row0 + li;
                if (li < nloc) {
                    if (grow == p && p != j) {
#pragma unroll
                        for (int c = 0; c < IB; ++c) a[r][c] = jr[c];
                    }
                    if (grow == j) {
#pragma unroll
                        for (int c = 0; c < IB; ++c) a[r][c] = prow[c];
                    }
                    if (grow > j) {
                        if (!sing) {
                            const E l = cmul(a[r][0], ip);
                            a[r][0] = l;
                            // active window positions 1 .. nact, in groups of four: loads first, then the FMAs
                            static_for<0, IB / 4>([&](auto gc) {
                                constexpr int c0 = 4 * decltype(gc)::value + 1;
                                if (nact >= c0) {  // uniform
                                    E pr[4];
#pragma unroll
                                    for (int q = 0; q < 4; ++q) lds_e(prow_s + (unsigned)((c0 + q) * sizeof(E)), pr[q]);
                                    static_for<0, 4>([&](auto qc) {
                                        constexpr int c = c0 + decltype(qc)::value;
                                        if constexpr (c < IB) {
                                            if (c <= nact) a[r][c] = cfnma(a[r][c], l, pr[c - c0]);
                                        }
                                    });
                                }
                            });
                        }
                        const T v = cabs1(a[r][1]);
                        if (nact > 0 && v > myval) { myval = v; myli = li; }
                    }
                }
            }
            tick(5);
        }
        // ---- rotate the window: the finished column goes to the back
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const E first = a[r][0];
#pragma unroll
            for (int c = 0; c + 1 < IB; ++c) a[r][c] = a[r][c + 1];
            a[r][IB - 1] = first;
        }
    }
    if constexpr (TIMING) {
        if (tid == POLLW * 32 && dbg)
            for (int k = 0; k < 6; ++k) dbg[cta * 8 + k] = tph[k];
    }

    // ---- write back (multipliers are already scaled)
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const int li = tid + r * PANEL_NT;
        if (li < nloc) {
#pragma unroll
            for (int c = 0; c < IB; ++c)
                if (c < jb) A.set(row0 + li, c, a[r][c]);
        }
    }
    if (cta != 0) return;
    // ---- CTA 0 owns the top jb x jb block: inverses of its unit-lower and upper triangles (leaves of the TRSM
    //      recursion), and the net row permutation of this swap batch.
    if (tid < IB) {
#pragma unroll
        for (int c = 0; c < IB; ++c) topb[c * IB + tid] = a[0][c];
    }
    __syncthreads();
    E *xl = inv_s, *xu = inv_s + IB * IB;  // column-major jb x jb, ld = IB
    if (tid < jb) {
        const int cc = tid;  // column cc of inv(L): forward substitution on e_cc
        for (int i = 0; i < jb; ++i) xl[cc * IB + i] = mk((T)(i == cc ? 1 : 0), (T)0);
        for (int i = cc + 1; i < jb; ++i) {
            E s = mk((T)0, (T)0);
            for (int k = cc; k < i; ++k) s = cadd(s, cmul(topb[k * IB + i], xl[cc * IB + k]));
            xl[cc * IB + i] = mk(-s.x, -s.y);
        }
        for (int i = 0; i < jb; ++i) dinvL.set(i, cc, xl[cc * IB + i]);
    } else if (tid >= 32 && tid < 32 + jb) {
        const int cc = tid - 32;  // column cc of inv(U): back substitution on e_cc
        for (int i = 0; i < jb; ++i) xu[cc * IB + i] = mk((T)0, (T)0);
        xu[cc * IB + cc] = invp[cc];
        for (int i = cc - 1; i >= 0; --i) {
            E s = mk((T)0, (T)0);
            for (int k = i + 1; k <= cc; ++k) s = cadd(s, cmul(topb[k * IB + i], xu[cc * IB + k]));
            E q = cmul(s, invp[i]);
            xu[cc * IB + i] = mk(-q.x, -q.y);
        }
        for (int i = 0; i < jb; ++i) dinvU.set(i, cc, xu[cc * IB + i]);
    } else if (warp == 2) {
        net_permutation(piv, jb, j0, perm, lane);
    }
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
static inline int split(int w) {
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
    static bool configured = false;
    if (!configured) {
        HP_CUDA(cudaFuncSetAttribute(inv_double_kernel<V>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = true;
    }
    ProfCat pc(PROF_OTHER);
    const bool prof = prof_enabled();
    if (prof) prof_begin(st, 0.0);
    inv_double_kernel<V><<<dim3(ceil_div(w, INV_RS), 2), INV_NT, smem, st>>>(A.sub(c0, c0), h, w, La, Lb, Lo, Ua, Ub, Uo);
    if (prof) prof_end(st);
    HP_LAUNCHED();
    return 0;
}

template <class V, int RPT>
static int launch_panel_reg(cudaStream_t st, V Asub, int m, int w, int c0, int rpc, int G, int *ipiv, int *info_dev,
                            LuWork<V> &wk, V dl, V du, int *perm) {
    typedef typename V::elem_t E;
    const size_t smem = 3 * (size_t)IB * IB * sizeof(E);
    auto kern = panel_reg_kernel<V, RPT>;
    static bool configured = false;
    if (!configured) {
        HP_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = true;
    }
    unsigned ep = wk.ep_base;
    long long *dbg = nullptr;
    void *args[] = {&Asub, &m, &w, &c0, &rpc, &ipiv, &info_dev, &wk.slots, &ep, &dl, &du, &perm, &dbg};
    HP_CUDA(cudaLaunchCooperativeKernel((void *)kern, dim3(G), dim3(PANEL_NT), args, smem, st));
    wk.ep_base += (unsigned)w;
    return 0;
}

template <class V> struct PanelRows;  // rows one CTA of the register-resident kernel can hold
template <> struct PanelRows<ZView> { static constexpr int max_rpt = 1; };
template <> struct PanelRows<CView> { static constexpr int max_rpt = 2; };

template <class V> static int panel(cudaStream_t st, int n, V A, int c0, int w, int *ipiv, int *info_dev, LuWork<V> &wk) {
    typedef typename V::elem_t E;
    const int m = n - c0;
    int rpc = std::max(ceil_div(m, MAXG), PANEL_MINROWS);
    rpc = (int)round_up(rpc, 2);
    const int G = ceil_div(m, rpc);
    V Asub = A.sub(c0, c0);
    const int blk = c0 / IB;
    V dl = wk.dinvL[0].sub(0, (long)blk * IB), du = wk.dinvU[0].sub(0, (long)blk * IB);
    int *perm = wk.perm + (size_t)blk * PERM_STRIDE;
    {
        ProfCat pc(PROF_PANEL);
        const bool prof = prof_enabled();
        if (prof) prof_begin(st, 0.0);
        int rc = 0;
        if (rpc <= PANEL_NT) {
            rc = launch_panel_reg<V, 1>(st, Asub, m, w, c0, rpc, G, ipiv, info_dev, wk, dl, du, perm);
        } else if (rpc <= PanelRows<V>::max_rpt * PANEL_NT) {
            rc = launch_panel_reg<V, PanelRows<V>::max_rpt>(st, Asub, m, w, c0, rpc, G, ipiv, info_dev, wk, dl, du, perm);
        } else {
            // taller than the register file allows: the shared-memory kernel with a counter barrier
            const size_t smem = ((size_t)IB * rpc + 2 * IB * IB) * sizeof(E);
            auto kern = panel_lu_kernel<V>;
            static size_t configured = 0;
            if (smem > configured) {
                HP_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                configured = smem;
            }
            int m_ = m, w_ = w, c0_ = c0, rpc_ = rpc;
            unsigned base = wk.bar_base;
            void *args[] = {&Asub, &m_, &w_, &c0_, &rpc_, &ipiv, &info_dev, &wk.cand_val, &wk.cand_row, &wk.cand_data,
                            &wk.jrow, &wk.counter, &base, &dl, &du, &perm};
            cudaError_t e = cudaLaunchCooperativeKernel((void *)kern, dim3(G), dim3(PANEL_NT), args, smem, st);
            if (e != cudaSuccess) rc = hp::cuda_fail(e, __FILE__, __LINE__);
            wk.bar_base += (unsigned)G * (unsigned)w;
        }
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
    copy_block_kernel<V><<<ceil_div((long)rows * cols, 256), 256, 0, st>>>(Src, Dst, rows, cols);
    HP_LAUNCHED();
    return 0;
}
// does the SB-aligned block starting at d0 have a kept full inverse, and is [d0, d0 + s) exactly that block?
static inline bool is_big_block(int n, int d0, int s) { return d0 % SB == 0 && s > LEAF && s == std::min(SB, n - d0); }
template <class V> static V binv_of(const V &tab, long sbld, int d0) { return tab.sub(0, (long)(d0 / SB) * sbld); }

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
template <class V> struct IsPlanar { static constexpr bool value = false; };
template <> struct IsPlanar<CView> { static constexpr bool value = true; };

// B <- inv * B for an SB block: out of place into the scratch, then copied back.  acc (complex64 solves): the kept inverse
// has its LEAF-diagonal blocks zeroed; those are applied from the dinv table with the 3xTF32 kernel.
template <class V>
static int big_leaf(cudaStream_t st, const V &binv, const V *dtab, int d0, int s, V B, int ncols, LuWork<V> &wk, bool acc) {
    const long cap = std::max<long>(wk.n, 256);
    for (long c = 0; c < ncols; c += cap) {
        const int nc = (int)std::min<long>(cap, ncols - c);
        V Bc = B.sub(0, c), T = wk.tmp;
        if (acc && IsPlanar<V>::value) {
            HP_TRY(diag_blocks_product(st, dtab, d0, s, Bc, nc, T));
            HP_TRY(gemm(st, s, nc, s, 1.0, binv_of(binv, wk.sbld, d0), Bc, 1.0, T));
        } else {
            HP_TRY(gemm(st, s, nc, s, 1.0, binv_of(binv, wk.sbld, d0), Bc, 0.0, T));
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

// B <- L^-1 B, L = unit lower triangle of the s x s diagonal block of A at (d0,d0); B is s x ncols.  d0 is a multiple of
// LEAF, or s <= LEAF is a full block of its size class (or the ragged last block).
template <class V> static int trsm_lower(cudaStream_t st, V A, int d0, int s, V B, int ncols, LuWork<V> &wk, bool acc = false) {
    if (s <= 0 || ncols <= 0) return 0;
    if (s <= LEAF) return gemm_sel(acc, st, s, ncols, s, 1.0, dinv_of(wk.dinvL, d0, s), B, 0.0, B);
    if (wk.use_big && (acc || IsPlanar<V>::value) && is_big_block(wk.n, d0, s))
        return big_leaf(st, wk.binvL, wk.dinvL, d0, s, B, ncols, wk, acc);
    const int h = split(s);
    HP_TRY(trsm_lower(st, A, d0, h, B, ncols, wk, acc));
    HP_TRY(gemm(st, s - h, ncols, h, -1.0, A.sub(d0 + h, d0), B, 1.0, B.sub(h, 0)));
    return trsm_lower(st, A, d0 + h, s - h, B.sub(h, 0), ncols, wk, acc);
}

// B <- U^-1 B, U = upper triangle (with diagonal) of the s x s diagonal block of A at (d0,d0)
template <class V> static int trsm_upper(cudaStream_t st, V A, int d0, int s, V B, int ncols, LuWork<V> &wk, bool acc = false) {
    if (s <= 0 || ncols <= 0) return 0;
    if (s <= LEAF) return gemm_sel(acc, st, s, ncols, s, 1.0, dinv_of(wk.dinvU, d0, s), B, 0.0, B);
    if (wk.use_big && (acc || IsPlanar<V>::value) && is_big_block(wk.n, d0, s))
        return big_leaf(st, wk.binvU, wk.dinvU, d0, s, B, ncols, wk, acc);
    const int h = split(s);
    HP_TRY(trsm_upper(st, A, d0 + h, s - h, B.sub(h, 0), ncols, wk, acc));
    HP_TRY(gemm(st, h, ncols, s - h, -1.0, A.sub(d0, d0 + h), B.sub(h, 0), 1.0, B));
    return trsm_upper(st, A, d0, h, B, ncols, wk, acc);
}

// Full inverses of the unit-lower and upper triangles of the SB block [c0, c0 + s): triangular solves on the identity with
// the LEAF-level recursion (the block's own big leaf does not exist yet).
// What the factorisation itself does not need (for complex128 both inverses: its U12 solves keep the LEAF-level recursion,
// whose GEMMs run at full FP64 rate; for complex64 the upper one) is built on a side stream, under the rest of the LU.
static cudaStream_t side_stream() {
    static cudaStream_t s = nullptr;
    if (!s && cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) s = nullptr;
    return s;
}
// `to` waits for everything enqueued on `from` so far
static int stream_follow(cudaStream_t from, cudaStream_t to) {
    cudaEvent_t e;
    HP_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    cudaError_t r1 = cudaEventRecord(e, from), r2 = cudaStreamWaitEvent(to, e, 0);
    cudaEventDestroy(e);
    HP_CUDA(r1);
    HP_CUDA(r2);
    return 0;
}

template <class V> static int build_binv(cudaStream_t st, V A, int c0, int s, LuWork<V> &wk) {
    ProfCat pc(PROF_OTHER);
    V XL = binv_of(wk.binvL, wk.sbld, c0), XU = binv_of(wk.binvU, wk.sbld, c0);
    cudaStream_t sd = side_stream();
    if (!sd) sd = st;
    if (sd != st) HP_TRY(stream_follow(st, sd));
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
    wk.side_used = (sd != st);
    return rc;
}

template <class V> static int getrf_rec(cudaStream_t st, int n, V A, int c0, int c1, int *ipiv, int *info_dev, LuWork<V> &wk) {
    const int w = c1 - c0;
    if (w <= IB) return panel(st, n, A, c0, w, ipiv, info_dev, wk);
    const int h = split(w), mid = c0 + h;
    HP_TRY(getrf_rec(st, n, A, c0, mid, ipiv, info_dev, wk));
    {
        ProfCat pc(PROF_LU_TRSM);
        HP_TRY(trsm_lower(st, A, c0, h, A.sub(c0, mid), c1 - mid, wk));
    }
    {
        ProfCat pc(PROF_LU_GEMM);
        HP_TRY(gemm(st, n - mid, c1 - mid, h, -1.0, A.sub(mid, c0), A.sub(c0, mid), 1.0, A.sub(mid, mid)));
    }
    HP_TRY(getrf_rec(st, n, A, mid, c1, ipiv, info_dev, wk));
    // the node's diagonal block is final: keep its inverse for the triangular solves further up / in getrs
    if (w <= LEAF) HP_TRY(inv_double(st, A, c0, h, w, wk));
    if (is_big_block(n, c0, w)) HP_TRY(build_binv(st, A, c0, w, wk));
    return 0;
}

template <class V> int getrf(cudaStream_t st, int n, V A, int *ipiv, int *info_dev, LuWork<V> &wk) {
    if (n <= 0) return 0;
    HP_CUDA(cudaMemsetAsync(wk.counter, 0, sizeof(unsigned), st));
    HP_CUDA(cudaMemsetAsync(wk.slots, 0, sizeof(unsigned long long) * LL_WORDS, st));
    wk.bar_base = 0;
    wk.ep_base = 0;
    wk.use_big = true;
    wk.side_used = false;
    HP_TRY(getrf_rec(st, n, A, 0, n, ipiv, info_dev, wk));
    if (wk.side_used) HP_TRY(stream_follow(side_stream(), st));  // join: the kept inverses are complete
    if (IsPlanar<V>::value && n > LEAF) {
        // the solves apply the LEAF-diagonal blocks of the kept inverses separately, with FP32-class products
        ProfCat pc(PROF_OTHER);
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
    HP_TRY(laswp(st, B, 0, nrhs, 0, 0, wk.perm, 0, wk.nblk));
    // the right-hand sides and the solution are O(1): FP32-class diagonal-block products (3xTF32 for the complex64 type)
    HP_TRY(trsm_lower(st, A, 0, n, B, nrhs, wk, true));
    return trsm_upper(st, A, 0, n, B, nrhs, wk, true);
}

// Measurement aid (hprmat_probe_panel): `reps` back-to-back factorisations of the same m x IB panel (the data are garbage
// after the first one; only time is of interest) with the phase-timing variant of the register-resident kernel.
int probe_panel(cudaStream_t st, int m, int reps, float *A_re, float *A_im, long lda, void *work, double *us_per_panel,
                long long *phase_cycles_host) {
    LuWork<CView> wk;
    wk.carve(work, m);
    CView A(A_re, A_im, lda);
    int rpc = std::max(ceil_div(m, MAXG), PANEL_MINROWS);
    rpc = (int)round_up(rpc, 2);
    if (rpc > PANEL_NT) return -2;
    const int G = ceil_div(m, rpc);
    int *ipiv = nullptr, *info = nullptr;
    long long *dbg = nullptr;
    HP_CUDA(cudaMalloc((void **)&ipiv, sizeof(int) * (IB + 8)));
    info = ipiv + IB;
    HP_CUDA(cudaMalloc((void **)&dbg, sizeof(long long) * 8 * MAXG));
    HP_CUDA(cudaMemsetAsync(ipiv, 0, sizeof(int) * (IB + 8), st));
    HP_CUDA(cudaMemsetAsync(wk.slots, 0, sizeof(unsigned long long) * LL_WORDS, st));
    auto kern = panel_reg_kernel<CView, 1, true>;
    const size_t smem = 3 * (size_t)IB * IB * sizeof(float2);
    HP_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaEvent_t e0, e1;
    HP_CUDA(cudaEventCreate(&e0));
    HP_CUDA(cudaEventCreate(&e1));
    CView dl = wk.dinvL[0], du = wk.dinvU[0];
    int w = IB, c0 = 0;
    for (int it = 0; it <= reps; ++it) {
        if (it == 1) HP_CUDA(cudaEventRecord(e0, st));
        unsigned ep = wk.ep_base;
        void *args[] = {&A, &m, &w, &c0, &rpc, &ipiv, &info, &wk.slots, &ep, &dl, &du, &wk.perm, &dbg};
        HP_CUDA(cudaLaunchCooperativeKernel((void *)kern, dim3(G), dim3(PANEL_NT), args, smem, st));
        HP_LAUNCHED();
        wk.ep_base += IB;
    }
    HP_CUDA(cudaEventRecord(e1, st));
    HP_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    *us_per_panel = ms * 1e3 / reps;
    if (phase_cycles_host) HP_CUDA(cudaMemcpy(phase_cycles_host, dbg, sizeof(long long) * 8 * MAXG, cudaMemcpyDeviceToHost));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(ipiv);
    cudaFree(dbg);
    return 0;
}

template struct LuWork<CView>;
template int getrf<CView>(cudaStream_t, int, CView, int *, int *, LuWork<CView> &);
template int getrs<CView>(cudaStream_t, int, int, CView, CView, LuWork<CView> &);
template struct LuWork<ZView>;
template int getrf<ZView>(cudaStream_t, int, ZView, int *, int *, LuWork<ZView> &);
template int getrs<ZView>(cudaStream_t, int, int, ZView, ZView, LuWork<ZView> &);

}  // namespace hp
