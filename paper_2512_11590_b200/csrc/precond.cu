// precond.cu -- the FP64 block-diagonal preconditioner of the mixed-precision path and the kernels that move between the
// FP64 problem and the split-complex64 system the tensor cores factorise (reading R10).
//
// With K_d = blockdiag(K_1 .. K_Nc), K_c = the Nb x Nb diagonal block of C - E*I (kinetic + Bloch + centrifugal +
// threshold + V_cc, Eqs. 1, 3 of PAPER.md:73-97), the paper's Type 3 writes M = K_d (I + K_d^-1 V_coupling)
// (Eqs. 6-9).  The mixed path factorises  S = K_d^-1 (C - E*I) = I + K_d^-1 V_coupling  in complex64:
//     S[(c,i),(c',j)] = delta_cc' delta_ij + (1 - delta_cc') Kinv_c[i,j] V_cc'(r_j)
// and solves  S X = K_d^-1 B;  the FP64 residual of the refinement is always that of the ORIGINAL system
// (PAPER.md:151, 222), mapped through K_d^-1 before the low-precision correction solve.
#include "precond.cuh"
#include "lu.cuh"

namespace hp {

// ---------------------------------------------------------------------------------------------------- K_c^-1
// One CTA per channel: Gauss-Jordan inversion in place with partial pivoting (first row of maximal |re|+|im|), matrix
// column-major n x n in shared memory when it fits (n <= 118), else in its global output buffer (L2-resident).
constexpr int KI_NT = 512;

template <bool SMEM>
__global__ void __launch_bounds__(KI_NT) kinv_kernel(int nch, int nb, const double *__restrict__ hT,
                                                     const double *__restrict__ dg0, const double *__restrict__ ethr,
                                                     double energy, const double2 *__restrict__ V,
                                                     const double2 *__restrict__ W, long ldw, double2 *__restrict__ Kinv,
                                                     int *info) {
    extern __shared__ __align__(16) unsigned char smraw[];
    const int c = blockIdx.x, n = nb, tid = threadIdx.x;
    double2 *out = Kinv + (size_t)c * n * n;
    double2 *rowk = reinterpret_cast<double2 *>(smraw);  // [n] pivot row
    double2 *colk = rowk + n;                            // [n] pivot column
    int *piv = reinterpret_cast<int *>(colk + 2 * n);    // [n]  (after rowp, see the sweep)
    double2 *a = SMEM ? reinterpret_cast<double2 *>(piv + ((n + 3) & ~3)) : out;  // compile-time: shared-space accesses
    __shared__ double red_v[KI_NT / 32];
    __shared__ int red_i[KI_NT / 32];

    for (int idx = tid; idx < n * n; idx += KI_NT) {
        const int i = idx % n, j = idx / n;
        double2 v = make_double2(hT[(size_t)j * n + i], 0.0);
        if (W) {  // non-local potentials: the full diagonal block of W is added (same rounding order as the assembly)
            const double2 wv = W[((size_t)c * n + j) * ldw + (size_t)c * n + i];
            const double base = (i == j) ? __dadd_rn(dg0[(size_t)c * n + i], __dsub_rn(ethr[c], energy)) : v.x;
            v.x = __dadd_rn(base, wv.x);
            v.y = wv.y;
        } else if (i == j) {
            const double2 vd = V[((size_t)i * nch + c) * nch + c];
            const double d2 = __dadd_rn(dg0[(size_t)c * n + i], __dsub_rn(ethr[c], energy));
            v.x = __dadd_rn(d2, vd.x);
            v.y = vd.y;
        }
        a[idx] = v;
    }
    __syncthreads();

    // Per step k (the kernel is bound by its instruction count, so the sweep over the matrix is kept branch-free):
    //  (A) warp-level arg-max of column k, barrier, every thread finishes the reduction itself -> pivot row p;
    //  (B1) stage old row k, old row p, column k; barrier;  (B2) exchange rows k and p in place and in the staged column; barrier;
    //  (C) a_ij -= c_i r_j (r_j = pivot row / pv) for every i and every j != k, one multiply-add chain per element with no case
    //       distinction; the owner of row k then overwrites it with r_j; column k is written separately: -c_i / pv, and 1 / pv
    //       on the diagonal;  barrier.
    double2 *rowp = rowk + 2 * n;  // [n] old row p (the pivot row before scaling); rowk: old row k; colk: column k
    for (int k = 0; k < n; ++k) {
        // (A)
        double bv = -1.0;
        int bi = -1;
        for (int i = k + tid; i < n; i += KI_NT) {
            const double v = cabs1(a[(size_t)k * n + i]);
            if (v > bv) { bv = v; bi = i; }
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const double ov = __shfl_down_sync(0xffffffffu, bv, off);
            const int oi = __shfl_down_sync(0xffffffffu, bi, off);
            if (ov > bv || (ov == bv && oi >= 0 && (bi < 0 || oi < bi))) { bv = ov; bi = oi; }
        }
        if ((tid & 31) == 0) { red_v[tid >> 5] = bv; red_i[tid >> 5] = bi; }
        __syncthreads();
        bv = red_v[0];
        bi = red_i[0];
        const int nw = min(KI_NT / 32, (n - k + 31) / 32);  // warps that had rows to look at
        for (int w = 1; w < nw; ++w) {
            const double ov = red_v[w];
            const int oi = red_i[w];
            if (ov > bv || (ov == bv && oi >= 0 && (bi < 0 || oi < bi))) { bv = ov; bi = oi; }
        }
        const int p = bi < 0 ? k : bi;  // (bi < 0: NaN column; reported as singular below)
        if (tid == 0) {
            piv[k] = p;
            if (!(bv > 0.0)) atomicCAS(info, 0, c * n + k + 1);
        }
        // (B1)
        for (int j = tid; j < n; j += KI_NT) {
            rowk[j] = a[(size_t)j * n + k];
            rowp[j] = a[(size_t)j * n + p];
            colk[j] = a[(size_t)k * n + j];
        }
        __syncthreads();
        const double2 pv = rowp[k];
        const bool sing = (pv.x == 0.0 && pv.y == 0.0);
        const double2 ip = sing ? make_double2(0.0, 0.0) : crecip_fast(pv);
        // (B2)
        if (p != k)
            for (int j = tid; j < n; j += KI_NT) {
                a[(size_t)j * n + k] = rowp[j];
                a[(size_t)j * n + p] = rowk[j];
            }
        if (tid == 0 && p != k) {  // column k with its entries k and p exchanged
            colk[p] = rowk[k];
            colk[k] = rowp[k];
        }
        __syncthreads();
        // (C) 32 rows x 16 columns of threads; the column-k values of a thread's rows sit in registers
        {
            const int ti = tid & 31, tj = tid >> 5;
            constexpr int RC = 4;  // rows ti + 32 a, a < RC, cached (covers n <= 128)
            double2 ck[RC];
#pragma unroll
            for (int r = 0; r < RC; ++r) ck[r] = (ti + 32 * r < n) ? colk[ti + 32 * r] : make_double2(0.0, 0.0);
            for (int j = tj; j < n; j += KI_NT / 32) {
                double2 *col = a + (size_t)j * n;
                if (j == k) {  // warp-uniform
                    for (int i = ti; i < n; i += 32) {
                        const double2 ci = colk[i];
                        col[i] = (i == k) ? ip : cmul(make_double2(-ci.x, -ci.y), ip);
                    }
                    continue;
                }
                const double2 rj = cmul(rowp[j], ip);
#pragma unroll
                for (int r = 0; r < RC; ++r)
                    if (ti + 32 * r < n) col[ti + 32 * r] = cfnma(col[ti + 32 * r], ck[r], rj);
                for (int i = ti + 32 * RC; i < n; i += 32) col[i] = cfnma(col[i], colk[i], rj);
                if (ti == (k & 31)) col[k] = rj;  // row k, by the thread that has just swept over it: the scaled pivot row
            }
        }
        __syncthreads();
    }
    // undo the row interchanges: columns of the inverse, in reverse order.  In shared memory the exchanges are applied to an
    // index array (one thread, n steps) and the columns are permuted on their way out; in place otherwise.
    if (SMEM) {
        __shared__ int cperm[128];              // the shared-memory path holds n <= 112
        if (tid == 0) {
            for (int j = 0; j < n; ++j) cperm[j] = j;
            for (int k = n - 1; k >= 0; --k) {
                const int p = piv[k];
                const int t = cperm[k];
                cperm[k] = cperm[p];
                cperm[p] = t;
            }
        }
        __syncthreads();
        for (int idx = tid; idx < n * n; idx += KI_NT) {
            const int i = idx % n, j = idx / n;
            out[idx] = a[(size_t)cperm[j] * n + i];
        }
    } else {
        for (int k = n - 1; k >= 0; --k) {
            const int p = piv[k];
            if (p != k) {
                for (int i = tid; i < n; i += KI_NT) {
                    const double2 t = a[(size_t)k * n + i];
                    a[(size_t)k * n + i] = a[(size_t)p * n + i];
                    a[(size_t)p * n + i] = t;
                }
            }
            __syncthreads();
        }
    }
}

int precond_invert(cudaStream_t st, const StructTables &t, double energy, const double2 *V, double2 *Kinv, int *info_dev,
                   const double2 *W, long ldw) {
    const int n = t.nb;
    const size_t small = sizeof(double2) * 3 * n + sizeof(int) * ((n + 3) & ~3);
    const size_t full = small + sizeof(double2) * (size_t)n * n;
    const int use_smem = full <= 200 * 1024 && n <= 128;  // (n <= 128: the kernel's column-permutation table)
    const size_t smem = use_smem ? full : small;
    if (use_smem) {
        static SmemCfg cfg;
        if (smem > 48 * 1024) HP_TRY(configure_smem(cfg, kinv_kernel<true>, smem));
        kinv_kernel<true><<<t.nch, KI_NT, smem, st>>>(t.nch, n, t.hT, t.dg0, t.ethr, energy, V, W, ldw, Kinv, info_dev);
    } else {
        kinv_kernel<false><<<t.nch, KI_NT, smem, st>>>(t.nch, n, t.hT, t.dg0, t.ethr, energy, V, W, ldw, Kinv, info_dev);
    }
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- assemble S
// Thread = one row (c,i) x one mesh column j x SA_CC consecutive column channels c': loads Kinv_c[i,j] once and writes
// SA_CC entries, each store instruction of a warp covering 128 contiguous bytes of a plane.
constexpr int SA_NT = 256, SA_CC = 8;

__global__ void __launch_bounds__(SA_NT) assemble_s_kernel(int nch, int nb, const double2 *__restrict__ Kinv,
                                                           const double2 *__restrict__ V, float *__restrict__ Sre,
                                                           float *__restrict__ Sim, long ld) {
    const int N = nch * nb;
    const int row = blockIdx.x * SA_NT + threadIdx.x;
    if (row >= N) return;
    const int c = row / nb, i = row - c * nb;
    const int j = blockIdx.y;
    const int cc0 = blockIdx.z * SA_CC;
    const double2 kij = Kinv[((size_t)c * nb + j) * nb + i];
#pragma unroll
    for (int e = 0; e < SA_CC; ++e) {
        const int c2 = cc0 + e;
        if (c2 >= nch) break;
        float re, im;
        if (c2 == c) {
            re = (i == j) ? 1.f : 0.f;
            im = 0.f;
        } else {
            const double2 v = V[((size_t)j * nch + c2) * nch + c];
            re = (float)(kij.x * v.x - kij.y * v.y);
            im = (float)(kij.x * v.y + kij.y * v.x);
        }
        const size_t off = (size_t)(c2 * nb + j) * ld + row;
        Sre[off] = re;
        Sim[off] = im;
    }
}

// The same with FOUR consecutive rows per thread (nb a multiple of 4, so that they share their channel; planes and leading
// dimension 16-byte aligned): every store instruction of a warp covers 512 contiguous bytes of a plane instead of 128 -- the
// write stream of 8 N^2 bytes is what this kernel is.
__global__ void __launch_bounds__(SA_NT) assemble_s4_kernel(int nch, int nb, const double2 *__restrict__ Kinv,
                                                            const double2 *__restrict__ V, float *__restrict__ Sre,
                                                            float *__restrict__ Sim, long ld) {
    const int N = nch * nb;
    const int row = 4 * (blockIdx.x * SA_NT + threadIdx.x);
    if (row >= N) return;
    const int c = row / nb, i = row - c * nb;
    const int j = blockIdx.y;
    const int cc0 = blockIdx.z * SA_CC;
    const double2 *kp = Kinv + ((size_t)c * nb + j) * nb + i;
    const double2 k0 = kp[0], k1 = kp[1], k2 = kp[2], k3 = kp[3];
#pragma unroll
    for (int e = 0; e < SA_CC; ++e) {
        const int c2 = cc0 + e;
        if (c2 >= nch) break;
        float4 re, im;
        if (c2 == c) {
            re = make_float4(i == j ? 1.f : 0.f, i + 1 == j ? 1.f : 0.f, i + 2 == j ? 1.f : 0.f, i + 3 == j ? 1.f : 0.f);
            im = make_float4(0.f, 0.f, 0.f, 0.f);
        } else {
            const double2 v = V[((size_t)j * nch + c2) * nch + c];
            re = make_float4((float)(k0.x * v.x - k0.y * v.y), (float)(k1.x * v.x - k1.y * v.y),
                             (float)(k2.x * v.x - k2.y * v.y), (float)(k3.x * v.x - k3.y * v.y));
            im = make_float4((float)(k0.x * v.y + k0.y * v.x), (float)(k1.x * v.y + k1.y * v.x),
                             (float)(k2.x * v.y + k2.y * v.x), (float)(k3.x * v.y + k3.y * v.x));
        }
        const size_t off = (size_t)(c2 * nb + j) * ld + row;
        *reinterpret_cast<float4 *>(Sre + off) = re;
        *reinterpret_cast<float4 *>(Sim + off) = im;
    }
}

int precond_assemble(cudaStream_t st, const StructTables &t, const double2 *Kinv, const double2 *V, CView S) {
    const int N = t.nch * t.nb;
    if (t.nb % 4 == 0 && S.ld % 4 == 0 && (((uintptr_t)S.re | (uintptr_t)S.im) & 15) == 0) {
        dim3 grid4(ceil_div(N / 4, SA_NT), t.nb, ceil_div(t.nch, SA_CC));
        assemble_s4_kernel<<<grid4, SA_NT, 0, st>>>(t.nch, t.nb, Kinv, V, S.re, S.im, S.ld);
        HP_LAUNCHED();
        return 0;
    }
    dim3 grid(ceil_div(N, SA_NT), t.nb, ceil_div(t.nch, SA_CC));
    assemble_s_kernel<<<grid, SA_NT, 0, st>>>(t.nch, t.nb, Kinv, V, S.re, S.im, S.ld);
    HP_LAUNCHED();
    return 0;
}

// FP64 variants (the preconditioned FP64 factorisation, ctx.cu solve_fp64_precond): same entries, interleaved complex128.
__global__ void __launch_bounds__(SA_NT) assemble_s_z_kernel(int nch, int nb, const double2 *__restrict__ Kinv,
                                                             const double2 *__restrict__ V, double2 *__restrict__ S, long ld) {
    const int N = nch * nb;
    const int row = blockIdx.x * SA_NT + threadIdx.x;
    if (row >= N) return;
    const int c = row / nb, i = row - c * nb;
    const int j = blockIdx.y;
    const int cc0 = blockIdx.z * SA_CC;
    const double2 kij = Kinv[((size_t)c * nb + j) * nb + i];
#pragma unroll
    for (int e = 0; e < SA_CC; ++e) {
        const int c2 = cc0 + e;
        if (c2 >= nch) break;
        double2 out;
        if (c2 == c) {
            out = make_double2((i == j) ? 1.0 : 0.0, 0.0);
        } else {
            const double2 v = V[((size_t)j * nch + c2) * nch + c];
            out = make_double2(kij.x * v.x - kij.y * v.y, kij.x * v.y + kij.y * v.x);
        }
        S[(size_t)(c2 * nb + j) * ld + row] = out;
    }
}

int precond_assemble_z(cudaStream_t st, const StructTables &t, const double2 *Kinv, const double2 *V, ZView S) {
    const int N = t.nch * t.nb;
    dim3 grid(ceil_div(N, SA_NT), t.nb, ceil_div(t.nch, SA_CC));
    assemble_s_z_kernel<<<grid, SA_NT, 0, st>>>(t.nch, t.nb, Kinv, V, S.p, S.ld);
    HP_LAUNCHED();
    return 0;
}

__global__ void __launch_bounds__(256) rhs_s_z_kernel(int nch, int nb, const double2 *__restrict__ Kinv,
                                                      const double *__restrict__ fa, double2 *__restrict__ B, long ld) {
    const long N = (long)nch * nb;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= N * nch) return;
    const int q = (int)(idx / N);
    const int row = (int)(idx - (long)q * N);
    const int c = row / nb, i = row - c * nb;
    double sr = 0.0, si = 0.0;
    if (c == q) {
        const double2 *k = Kinv + (size_t)c * nb * nb + i;
        for (int j = 0; j < nb; ++j) {
            const double2 v = k[(size_t)j * nb];
            sr = fma(v.x, fa[j], sr);
            si = fma(v.y, fa[j], si);
        }
    }
    B[(size_t)q * ld + row] = make_double2(sr, si);
}

int precond_rhs_z(cudaStream_t st, const StructTables &t, const double2 *Kinv, ZView B) {
    const long tot = (long)t.nch * t.nb * t.nch;
    rhs_s_z_kernel<<<ceil_div(tot, 256), 256, 0, st>>>(t.nch, t.nb, Kinv, t.fa, B.p, B.ld);
    HP_LAUNCHED();
    return 0;
}

// Non-local potentials: S = K_d^-1 (C - E I) with full blocks.  Block row c of S is Kinv_c times block row c of W for the
// off-diagonal blocks and the identity on the diagonal block.  The products run on the FP64 tensor cores, one column chunk
// of nch columns at a time (nch batched nb x nch x nb GEMMs into the N x nch scratch T), and this kernel demotes the chunk
// into the float planes, writing the identity where the column lies in the row's own channel.
__global__ void __launch_bounds__(256) demote_offdiag_kernel(int nch, int nb, int j0, int w, const double2 *__restrict__ T,
                                                             long ldt, float *__restrict__ Sre, float *__restrict__ Sim,
                                                             long ld) {
    const long N = (long)nch * nb;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= N * w) return;
    const int q = (int)(idx / N);
    const long row = idx - (long)q * N;
    const int col = j0 + q;
    float re, im;
    if (row / nb == col / nb) {
        re = (row == col) ? 1.f : 0.f;
        im = 0.f;
    } else {
        const double2 v = T[(long)q * ldt + row];
        re = (float)v.x;
        im = (float)v.y;
    }
    Sre[(long)col * ld + row] = re;
    Sim[(long)col * ld + row] = im;
}

int precond_assemble_nonlocal(cudaStream_t st, const StructTables &t, const double2 *Kinv, const double2 *W, long ldw, CView S,
                              double2 *T, long ldt) {
    const int nch = t.nch, nb = t.nb, N = nch * nb;
    for (int j0 = 0; j0 < N; j0 += nch) {
        const int w = std::min(nch, N - j0);
        HP_TRY(zgemm_batched(st, nb, w, nb, 1.0, Kinv, nb, (long)nb * nb, W + (long)j0 * ldw, ldw, nb, 0.0, T, ldt, nb, nch));
        demote_offdiag_kernel<<<ceil_div((long)N * w, 256), 256, 0, st>>>(nch, nb, j0, w, T, ldt, S.re, S.im, S.ld);
        HP_LAUNCHED();
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------------- right-hand side
// (K_d^-1 B)[(c,i),c'] = delta_cc' sum_j Kinv_c[i,j] fa_j, demoted to the split-complex64 right-hand side block.
__global__ void __launch_bounds__(256) rhs_s_kernel(int nch, int nb, const double2 *__restrict__ Kinv,
                                                    const double *__restrict__ fa, float *__restrict__ Bre,
                                                    float *__restrict__ Bim, long ld) {
    const long N = (long)nch * nb;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= N * nch) return;
    const int q = (int)(idx / N);
    const int row = (int)(idx - (long)q * N);
    const int c = row / nb, i = row - c * nb;
    float re = 0.f, im = 0.f;
    if (c == q) {
        double sr = 0.0, si = 0.0;
        const double2 *k = Kinv + (size_t)c * nb * nb + i;
        for (int j = 0; j < nb; ++j) {
            const double2 v = k[(size_t)j * nb];
            sr = fma(v.x, fa[j], sr);
            si = fma(v.y, fa[j], si);
        }
        re = (float)sr;
        im = (float)si;
    }
    Bre[(size_t)q * ld + row] = re;
    Bim[(size_t)q * ld + row] = im;
}

int precond_rhs(cudaStream_t st, const StructTables &t, const double2 *Kinv, CView B) {
    const long tot = (long)t.nch * t.nb * t.nch;
    rhs_s_kernel<<<ceil_div(tot, 256), 256, 0, st>>>(t.nch, t.nb, Kinv, t.fa, B.re, B.im, B.ld);
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- precision moves
// complex128 (interleaved) -> split complex64
__global__ void __launch_bounds__(256) demote_kernel(long rows, int cols, const double2 *__restrict__ Z, long ldz,
                                                     float *__restrict__ re, float *__restrict__ im, long ld) {
    const long tot = rows * cols;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long q = idx / rows, r = idx - q * rows;
        const double2 z = Z[q * ldz + r];
        re[q * ld + r] = (float)z.x;
        im[q * ld + r] = (float)z.y;
    }
}

int demote(cudaStream_t st, long rows, int cols, const double2 *Z, long ldz, CView D) {
    const long tot = rows * cols;
    if (tot <= 0) return 0;
    const int grid = (int)std::min<long>(ceil_div(tot, 256), 148L * 8);
    demote_kernel<<<grid, 256, 0, st>>>(rows, cols, Z, ldz, D.re, D.im, D.ld);
    HP_LAUNCHED();
    return 0;
}

// X <- (accumulate ? X : 0) + D with D split complex64 (PAPER.md:220 c2z, :225 add_correction, fused);
// norms[0] = max|D|, norms[1] = max|X_new| (moduli; pre-zeroed here)
__global__ void __launch_bounds__(256) promote_add_kernel(long rows, int cols, double2 *__restrict__ X, long ldx,
                                                          const float *__restrict__ re, const float *__restrict__ im, long ld,
                                                          int accumulate, double *norms, const int *gate) {
    __shared__ double shred[32];
    if (gate != nullptr && *gate != 0) return;  // the refinement has already stopped: this step must not touch X
    double md = 0.0, mx = 0.0;
    const long tot = rows * cols;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long q = idx / rows, r = idx - q * rows;
        const double dr = (double)re[q * ld + r], di = (double)im[q * ld + r];
        double2 x = accumulate ? X[q * ldx + r] : make_double2(0.0, 0.0);
        x.x += dr;
        x.y += di;
        X[q * ldx + r] = x;
        md = fmax(md, sqrt(dr * dr + di * di));
        mx = fmax(mx, sqrt(x.x * x.x + x.y * x.y));
    }
    // block maxima (same reduction shape as structured.cu's)
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        md = fmax(md, __shfl_xor_sync(0xffffffffu, md, off));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { shred[warp] = md; shred[8 + warp] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { md = fmax(md, shred[w]); mx = fmax(mx, shred[8 + w]); }
        atomicMax(reinterpret_cast<unsigned long long *>(norms), (unsigned long long)__double_as_longlong(md));
        atomicMax(reinterpret_cast<unsigned long long *>(norms + 1), (unsigned long long)__double_as_longlong(mx));
    }
}

int promote_add(cudaStream_t st, long rows, int cols, double2 *X, long ldx, CView D, bool accumulate, double *norms_dev,
                const int *gate_dev) {
    HP_CUDA(cudaMemsetAsync(norms_dev, 0, 2 * sizeof(double), st));
    const long tot = rows * cols;
    if (tot <= 0) return 0;
    const int grid = (int)std::min<long>(ceil_div(tot, 256), 148L * 8);
    promote_add_kernel<<<grid, 256, 0, st>>>(rows, cols, X, ldx, D.re, D.im, D.ld, accumulate ? 1 : 0, norms_dev, gate_dev);
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- Type 3 (literal)
// M = K_diag (I + K^-1 V) with K the REAL kinetic (+ Bloch) block shared by all channels, V(r_j) the
// Nc x Nc matrices of everything else on the mesh diagonal (potentials, centrifugal and threshold terms, -E), and the
// point-major Schur matrix of Eq. (8):  S[(i,a),(j,a')] = delta_ij delta_aa' + Kinv_ij V_aa'(r_j),  index (i*nch + a).
// Thread = (a, column (j,a')): loads V'_aa'(r_j) once and writes the nb entries of its column strip, each store of a warp
// covering 128 contiguous bytes of a plane.
__global__ void __launch_bounds__(128) assemble_type3_kernel(int nch, int nb, const double *__restrict__ KTinv,
                                                             const double *__restrict__ cf, const double *__restrict__ ethr,
                                                             double energy, const double2 *__restrict__ V,
                                                             float *__restrict__ Sre, float *__restrict__ Sim, long ld) {
    const int a = blockIdx.y * 128 + threadIdx.x;
    const long q = blockIdx.x;            // column (j, a')
    if (a >= nch) return;
    const int j = (int)(q / nch), a2 = (int)(q - (long)j * nch);
    double2 v = V[((long)j * nch + a2) * nch + a];  // V_{a a'}(r_j)
    if (a == a2) v.x += cf[(long)a * nb + j] + (ethr[a] - energy);
    float *re = Sre + q * ld + a, *im = Sim + q * ld + a;
    for (int i = 0; i < nb; ++i) {
        const double k = KTinv[(long)j * nb + i];
        re[(long)i * nch] = (float)(k * v.x + ((i == j && a == a2) ? 1.0 : 0.0));
        im[(long)i * nch] = (float)(k * v.y);
    }
}
int type3_assemble(cudaStream_t st, const StructTables &t, const double *KTinv, const double *cf, double energy, const double2 *V,
                   CView S) {
    const long N = (long)t.nch * t.nb;
    assemble_type3_kernel<<<dim3((unsigned)N, ceil_div(t.nch, 128)), 128, 0, st>>>(t.nch, t.nb, KTinv, cf, t.ethr, energy, V, S.re,
                                                                                  S.im, S.ld);
    HP_LAUNCHED();
    return 0;
}

// Eq. (9): b~[(i,a), c'] = (Kinv q2)_i delta_{a c'}   (g = Kinv q2 is energy-independent, computed at setup)
__global__ void __launch_bounds__(256) rhs_type3_kernel(int nch, int nb, const double *__restrict__ g, float *__restrict__ Bre,
                                                        float *__restrict__ Bim, long ld) {
    const long N = (long)nch * nb, tot = N * nch;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long c2 = idx / N, p = idx - c2 * N;
        const int i = (int)(p / nch), a = (int)(p - (long)i * nch);
        Bre[c2 * ld + p] = a == c2 ? (float)g[i] : 0.f;
        Bim[c2 * ld + p] = 0.f;
    }
}
int type3_rhs(cudaStream_t st, const StructTables &t, const double *g, CView B) {
    const long tot = (long)t.nch * t.nb * t.nch;
    rhs_type3_kernel<<<(int)std::min<long>(ceil_div(tot, 256), 148L * 8), 256, 0, st>>>(t.nch, t.nb, g, B.re, B.im, B.ld);
    HP_LAUNCHED();
    return 0;
}

// step 6 "transform solution back": X[(a,i), c'] <- x~[(i,a), c']  (point-major complex64 -> channel-major complex128);
// norms[1] = max|X|
__global__ void __launch_bounds__(256) promote_from_point_major_kernel(int nch, int nb, const float *__restrict__ re,
                                                                       const float *__restrict__ im, long ld,
                                                                       double2 *__restrict__ X, long ldx, double *norms) {
    __shared__ double shred[32];
    const long N = (long)nch * nb, tot = N * nch;
    double mx = 0.0;
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long c2 = idx / N, p = idx - c2 * N;
        const int i = (int)(p / nch), a = (int)(p - (long)i * nch);
        const double xr = (double)re[c2 * ld + p], xi = (double)im[c2 * ld + p];
        X[c2 * ldx + (long)a * nb + i] = make_double2(xr, xi);
        mx = fmax(mx, sqrt(xr * xr + xi * xi));
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, off));
    if ((threadIdx.x & 31) == 0) shred[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) mx = fmax(mx, shred[w]);
        atomicMax(reinterpret_cast<unsigned long long *>(norms + 1), (unsigned long long)__double_as_longlong(mx));
    }
}
int type3_promote(cudaStream_t st, const StructTables &t, CView Xs, double2 *X, long ldx, double *norms_dev) {
    HP_CUDA(cudaMemsetAsync(norms_dev, 0, 2 * sizeof(double), st));
    const long tot = (long)t.nch * t.nb * t.nch;
    promote_from_point_major_kernel<<<(int)std::min<long>(ceil_div(tot, 256), 148L * 8), 256, 0, st>>>(t.nch, t.nb, Xs.re, Xs.im,
                                                                                                       Xs.ld, X, ldx, norms_dev);
    HP_LAUNCHED();
    return 0;
}

}  // namespace hp
