// panel.cu -- panel factorisation of the blocked LU with partial pivoting (PAPER.md:125-131, Eq. 5; :127 "partial
// pivoting"): the register-resident cooperative kernel (fence-free epoch-tagged exchange between the CTAs), its
// shared-memory predecessor (kept for panels taller than the register file allows).  The factorisations whose pivots
// are verified to be the diagonal ones do not come here (toplu.cu).  See DESIGN.md section 6.
#include "panel.cuh"

#include <algorithm>


namespace hp {

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

// Inverses of the unit-lower and upper triangles of the factored top block (topb: column-major jb x jb, ld = IB, multipliers
// already scaled; invp[k] = 1/u_kk) -> dinvL / dinvU, the IB-level leaves of the triangular-solve recursion.  Threads
// 0 .. jb-1 do the columns of inv(L), threads 32 .. 32+jb-1 those of inv(U); inv_s is [2][IB][IB] scratch.
template <class V>
__device__ __forceinline__ void top_block_inverses(const typename V::elem_t *topb, const typename V::elem_t *invp,
                                                   typename V::elem_t *inv_s, int jb, V dinvL, V dinvU, int tid) {
    typedef typename V::elem_t E;
    typedef typename V::real_t T;
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
    }
}

template <class V, int RPT>
__global__ void __launch_bounds__(PANEL_NT, 1)
    panel_reg_kernel(V A, int m, int jb, int j0, int rpc, int *ipiv, int *info, unsigned long long *ll, unsigned ep_base,
                     V dinvL, V dinvU, int *perm) {
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

    E a[RPT][IB];
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
        const int li = tid + r * PANEL_NT;
#pragma unroll
        for (int c = 0; c < IB; ++c) a[r][c] = (li < nloc && c < jb) ? A.get(row0 + li, c) : mk((T)0, (T)0);
    }

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
    if (cta == 0) {
        // ---- CTA 0 owns the top jb x jb block: inverses of its unit-lower and upper triangles (leaves of the TRSM
        //      recursion), and the net row permutation of this swap batch.
        if (tid < IB) {
#pragma unroll
            for (int c = 0; c < IB; ++c) topb[c * IB + tid] = a[0][c];
        }
        __syncthreads();
        top_block_inverses<V>(topb, invp, inv_s, jb, dinvL, dinvU, tid);
        if (warp == 2) net_permutation(piv, jb, j0, perm, lane);
    }
}

template <class V, int RPT>
static int launch_panel_reg(cudaStream_t st, V Asub, int m, int w, int c0, int rpc, int G, int *ipiv, int *info_dev,
                            LuWork<V> &wk, V dl, V du, int *perm) {
    typedef typename V::elem_t E;
    const size_t smem = 3 * (size_t)IB * IB * sizeof(E);
    auto kern = panel_reg_kernel<V, RPT>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, smem));
    unsigned ep = wk.ep_base;
    void *args[] = {&Asub, &m, &w, &c0, &rpc, &ipiv, &info_dev, &wk.slots, &ep, &dl, &du, &perm};
    HP_CUDA(cudaLaunchCooperativeKernel((void *)kern, dim3(G), dim3(PANEL_NT), args, smem, st));
    wk.ep_base += (unsigned)w;
    return 0;
}

template <class V> struct PanelRows;  // rows one CTA of the register-resident kernel can hold
template <> struct PanelRows<ZView> { static constexpr int max_rpt = 1; };
template <> struct PanelRows<CView> { static constexpr int max_rpt = 2; };

template <class V>
int panel_launch(cudaStream_t st, V Asub, int m, int w, int c0, int *ipiv, int *info_dev, LuWork<V> &wk, V dl, V du, int *perm) {
    typedef typename V::elem_t E;
    int rpc = std::max(ceil_div(m, MAXG), PANEL_MINROWS);
    rpc = (int)round_up(rpc, 2);
    const int G = ceil_div(m, rpc);
    if (rpc <= PANEL_NT) return launch_panel_reg<V, 1>(st, Asub, m, w, c0, rpc, G, ipiv, info_dev, wk, dl, du, perm);
    if (rpc <= PanelRows<V>::max_rpt * PANEL_NT)
        return launch_panel_reg<V, PanelRows<V>::max_rpt>(st, Asub, m, w, c0, rpc, G, ipiv, info_dev, wk, dl, du, perm);
    // taller than the register file allows: the shared-memory kernel with a counter barrier
    const size_t smem = ((size_t)IB * rpc + 2 * IB * IB) * sizeof(E);
    auto kern = panel_lu_kernel<V>;
    static SmemCfg cfg;
    HP_TRY(configure_smem(cfg, kern, smem));
    unsigned base = wk.bar_base;
    void *args[] = {&Asub, &m, &w, &c0, &rpc, &ipiv, &info_dev, &wk.cand_val, &wk.cand_row, &wk.cand_data,
                    &wk.jrow, &wk.counter, &base, &dl, &du, &perm};
    HP_CUDA(cudaLaunchCooperativeKernel((void *)kern, dim3(G), dim3(PANEL_NT), args, smem, st));
    wk.bar_base += (unsigned)G * (unsigned)w;
    return 0;
}

template int panel_launch<CView>(cudaStream_t, CView, int, int, int, int *, int *, LuWork<CView> &, CView, CView, int *);
template int panel_launch<ZView>(cudaStream_t, ZView, int, int, int, int *, int *, LuWork<ZView> &, ZView, ZView, int *);

}  // namespace hp
