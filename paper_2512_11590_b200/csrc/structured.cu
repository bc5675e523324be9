// structured.cu -- the O(N^2)-and-below kernels of the structured R-matrix path: assembly of C - E*I (PAPER.md:87-99,
// Eqs. 3-4 with the diagonal terms of Eq. 1), the surface right-hand sides, the matrix-free FP64
// residual B - (C - E*I) X used by the iterative refinement, the update X += d with its
// convergence norms and the contraction R = (h2m/a) B^T X (PAPER.md:137 step 4).
// All of them are HBM- or L2-bound; none is a dense contraction large enough for tensor cores except the coupling part
// of the residual, which is kept on the FP64 pipe because it accumulates in double-double.
#include "structured.cuh"

namespace hp {

// ---------------------------------------------------------------------------------------------------- assembly
// One thread = one matrix row x ASM_CPT consecutive columns; consecutive threads = consecutive rows, so every store
// instruction of a warp writes 512 contiguous bytes of the column-major matrix.  Entry (row=(c1,i), col=(c2,j)):
//   c1 == c2:  hT[i,j]  (+ for i == j: ((dg0[c1,i]) + (E_c1 - E)) + V_c1c1(r_i), evaluated in exactly this order)
//   c1 != c2:  i == j ? V_c1c2(r_i) : 0
constexpr int ASM_NT = 256, ASM_CPT = 4;

__global__ void __launch_bounds__(ASM_NT) assemble_z_kernel(double2 *__restrict__ C, long ldc, int nch, int nb,
                                                            const double *__restrict__ hT, const double *__restrict__ dg0,
                                                            const double *__restrict__ ethr, double energy,
                                                            const double2 *__restrict__ V) {
    const int N = nch * nb;
    const int row = blockIdx.x * ASM_NT + threadIdx.x;
    if (row >= N) return;
    const int c1 = row / nb, i = row - c1 * nb;
    const int col0 = blockIdx.y * ASM_CPT;
#pragma unroll
    for (int e = 0; e < ASM_CPT; ++e) {
        const int col = col0 + e;
        if (col >= N) break;
        const int c2 = col / nb, j = col - c2 * nb;
        double2 v = make_double2(0.0, 0.0);
        if (c1 == c2) {
            v.x = hT[(long)j * nb + i];
            if (i == j) {
                const double2 vd = V[((long)i * nch + c2) * nch + c1];
                const double d2 = __dadd_rn(dg0[row], __dsub_rn(ethr[c1], energy));
                v.x = __dadd_rn(d2, vd.x);
                v.y = vd.y;
            }
        } else if (i == j) {
            v = V[((long)i * nch + c2) * nch + c1];
        }
        C[(long)col * ldc + row] = v;
    }
}

int assemble_z(cudaStream_t st, const StructTables &t, double energy, const double2 *V, double2 *C, long ldc) {
    const int N = t.nch * t.nb;
    dim3 grid(ceil_div(N, ASM_NT), ceil_div(N, ASM_CPT));
    assemble_z_kernel<<<grid, ASM_NT, 0, st>>>(C, ldc, t.nch, t.nb, t.hT, t.dg0, t.ethr, energy, V);
    HP_LAUNCHED();
    return 0;
}

// Non-local potentials (every block full): C = W + [kinetic + Bloch + centrifugal + threshold - E on the
// diagonal blocks], W the caller's N x N matrix of potential matrix elements.  Same thread mapping as assemble_z_kernel; the
// diagonal is evaluated as ((dg0 + (E_c - E)) + Re W_ii), the order of the local path.  Reads and writes 16 N^2 bytes each.
__global__ void __launch_bounds__(ASM_NT) assemble_nonlocal_kernel(double2 *__restrict__ C, long ldc, int nch, int nb,
                                                                   const double *__restrict__ hT,
                                                                   const double *__restrict__ dg0,
                                                                   const double *__restrict__ ethr, double energy,
                                                                   const double2 *__restrict__ W, long ldw) {
    const int N = nch * nb;
    const int row = blockIdx.x * ASM_NT + threadIdx.x;
    if (row >= N) return;
    const int c1 = row / nb, i = row - c1 * nb;
    const int col0 = blockIdx.y * ASM_CPT;
    double2 w[ASM_CPT];
#pragma unroll
    for (int e = 0; e < ASM_CPT; ++e)
        if (col0 + e < N) w[e] = W[(long)(col0 + e) * ldw + row];
#pragma unroll
    for (int e = 0; e < ASM_CPT; ++e) {
        const int col = col0 + e;
        if (col >= N) break;
        const int c2 = col / nb, j = col - c2 * nb;
        double2 v = w[e];
        if (c1 == c2) {
            if (i == j) v.x = __dadd_rn(__dadd_rn(dg0[row], __dsub_rn(ethr[c1], energy)), v.x);
            else v.x = __dadd_rn(hT[(long)j * nb + i], v.x);
        }
        C[(long)col * ldc + row] = v;
    }
}

int assemble_nonlocal(cudaStream_t st, const StructTables &t, double energy, const double2 *W, long ldw, double2 *C,
                      long ldc) {
    const int N = t.nch * t.nb;
    dim3 grid(ceil_div(N, ASM_NT), ceil_div(N, ASM_CPT));
    assemble_nonlocal_kernel<<<grid, ASM_NT, 0, st>>>(C, ldc, t.nch, t.nb, t.hT, t.dg0, t.ethr, energy, W, ldw);
    HP_LAUNCHED();
    return 0;
}

// ||W + diagonal-block terms||_inf (max row sum of moduli) without forming the matrix: one thread per row, a warp reads 512
// contiguous bytes of every column of W; columns are split over gridDim.y slices whose partial row sums meet in rowsum
// (pre-zeroed, N doubles).
__global__ void __launch_bounds__(256) nonlocal_rowsum_kernel(int nch, int nb, const double *__restrict__ hT,
                                                              const double *__restrict__ dg0,
                                                              const double *__restrict__ ethr, double energy,
                                                              const double2 *__restrict__ W, long ldw,
                                                              double *__restrict__ rowsum) {
    const int n = nch * nb;
    const int row = blockIdx.x * 256 + threadIdx.x;
    if (row >= n) return;
    const int c1 = row / nb, i = row - c1 * nb;
    const int per = (n + gridDim.y - 1) / gridDim.y;
    const int j0 = blockIdx.y * per, j1 = min(n, j0 + per);
    const double dterm = __dadd_rn(dg0[row], __dsub_rn(ethr[c1], energy));
    double s = 0.0;
#pragma unroll 4
    for (int col = j0; col < j1; ++col) {
        double2 v = W[(long)col * ldw + row];
        const int c2 = col / nb;
        if (c2 == c1) {
            const int j = col - c2 * nb;
            v.x = (i == j) ? __dadd_rn(dterm, v.x) : __dadd_rn(hT[(long)j * nb + i], v.x);
        }
        s += sqrt(v.x * v.x + v.y * v.y);
    }
    atomicAdd(rowsum + row, s);
}

int nonlocal_anorm(cudaStream_t st, const StructTables &t, double energy, const double2 *W, long ldw, double *rowsum_scratch,
                   double *out_dev) {
    const int n = t.nch * t.nb;
    HP_CUDA(cudaMemsetAsync(rowsum_scratch, 0, sizeof(double) * (size_t)n, st));
    dim3 grid(ceil_div(n, 256), std::max(1, std::min(64, n / 256)));
    nonlocal_rowsum_kernel<<<grid, 256, 0, st>>>(t.nch, t.nb, t.hT, t.dg0, t.ethr, energy, W, ldw, rowsum_scratch);
    HP_LAUNCHED();
    HP_CUDA(cudaMemsetAsync(out_dev, 0, sizeof(double), st));
    return maxabs_real(st, n, rowsum_scratch, out_dev);
}

// ---------------------------------------------------------------------------------------------------- right-hand side
__global__ void rhs_kernel(double2 *__restrict__ B, long ldb, int nch, int nb, const double *__restrict__ fa) {
    const long N = (long)nch * nb;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= N * nch) return;
    const int q = (int)(idx / N);
    const int row = (int)(idx - (long)q * N);
    const int c = row / nb, i = row - c * nb;
    B[(long)q * ldb + row] = make_double2(c == q ? fa[i] : 0.0, 0.0);
}

int build_rhs(cudaStream_t st, const StructTables &t, double2 *B, long ldb) {
    const long tot = (long)t.nch * t.nb * t.nch;
    rhs_kernel<<<ceil_div(tot, 256), 256, 0, st>>>(B, ldb, t.nch, t.nb, t.fa);
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- residual
// Double-double accumulation (TwoProduct by FMA + TwoSum): s + c carries the running sum to ~2^-104 relative, so the
// residual of the double matrix is exact to FP64 rounding of the result -- that is what lets one refinement step of the
// FP64 path, and the last steps of the mixed path, reach ~1e-15 on this ill-conditioned C.
__device__ __forceinline__ void dd_mac(double &s, double &c, double a, double b) {
    const double p = __dmul_rn(a, b);
    const double e = __fma_rn(a, b, -p);
    const double t = __dadd_rn(s, p);
    const double bb = __dsub_rn(t, s);
    const double err = __dadd_rn(__dsub_rn(s, __dsub_rn(t, bb)), __dsub_rn(p, bb));
    s = t;
    c = __dadd_rn(c, __dadd_rn(e, err));
}

constexpr int RES_QT = 4;    // right-hand sides per thread
constexpr int RES_NT = 128;

// Part 1: within-channel terms.  grid (nch, ceil(nrhs/QT)); thread = mesh point i of channel c = blockIdx.x.
//   acc[(c,i),q] = b[(c,i),q] - sum_{j != i} hT[i,j] X[(c,j),q] - Cdiag[(c,i)] X[(c,i),q]
// written as the (hi, lo) pair of the double-double sum.  Bx == nullptr: b = fa_i delta_cq (the surface RHS).
__global__ void __launch_bounds__(RES_NT) resid_channel_kernel(int nch, int nb, int nrhs, const double *__restrict__ hT,
                                                              const double *__restrict__ dg0,
                                                              const double *__restrict__ ethr, double energy,
                                                              const double *__restrict__ fa, const double2 *__restrict__ V,
                                                              const double2 *__restrict__ Bx, long ldb,
                                                              const double2 *__restrict__ X, long ldx,
                                                              double2 *__restrict__ Rhi, double2 *__restrict__ Rlo,
                                                              long ldr) {
    extern __shared__ __align__(16) unsigned char smraw[];
    double2 *Xs = reinterpret_cast<double2 *>(smraw);  // [QT][nb]
    const int c = blockIdx.x, q0 = blockIdx.y * RES_QT;
    const int nq = min(RES_QT, nrhs - q0);
    for (int idx = threadIdx.x; idx < RES_QT * nb; idx += RES_NT) {
        const int qq = idx / nb, j = idx - qq * nb;
        Xs[idx] = qq < nq ? X[(long)(q0 + qq) * ldx + (long)c * nb + j] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nb; i += RES_NT) {
        const long row = (long)c * nb + i;
        double sr[RES_QT], cr[RES_QT], si[RES_QT], ci[RES_QT];
#pragma unroll
        for (int qq = 0; qq < RES_QT; ++qq) {
            sr[qq] = si[qq] = cr[qq] = ci[qq] = 0.0;
            if (qq < nq) {
                if (Bx) {
                    const double2 b = Bx[(long)(q0 + qq) * ldb + row];
                    sr[qq] = b.x;
                    si[qq] = b.y;
                } else if (q0 + qq == c) {
                    sr[qq] = fa[i];
                }
            }
        }
        for (int j = 0; j < nb; ++j) {
            if (j == i) continue;
            const double t = -hT[(long)j * nb + i];
#pragma unroll
            for (int qq = 0; qq < RES_QT; ++qq) {
                const double2 x = Xs[qq * nb + j];
                dd_mac(sr[qq], cr[qq], t, x.x);
                dd_mac(si[qq], ci[qq], t, x.y);
            }
        }
        {
            const double2 vd = V[((long)i * nch + c) * nch + c];
            const double d2 = __dadd_rn(dg0[row], __dsub_rn(ethr[c], energy));
            const double dr = __dadd_rn(d2, vd.x), di = vd.y;
#pragma unroll
            for (int qq = 0; qq < RES_QT; ++qq) {
                const double2 x = Xs[qq * nb + i];
                dd_mac(sr[qq], cr[qq], -dr, x.x);
                dd_mac(sr[qq], cr[qq], di, x.y);
                dd_mac(si[qq], ci[qq], -dr, x.y);
                dd_mac(si[qq], ci[qq], -di, x.x);
            }
        }
#pragma unroll
        for (int qq = 0; qq < RES_QT; ++qq)
            if (qq < nq) {
                Rhi[(long)(q0 + qq) * ldr + row] = make_double2(sr[qq], si[qq]);
                Rlo[(long)(q0 + qq) * ldr + row] = make_double2(cr[qq], ci[qq]);
            }
    }
}

__device__ __forceinline__ void atomic_max_nonneg(double *addr, double v) {
    // non-negative doubles order like their bit patterns
    atomicMax(reinterpret_cast<unsigned long long *>(addr), (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ double block_max(double v, double *sh) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, off));
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    if (warp == 0) {
        v = lane < nw ? sh[lane] : 0.0;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, off));
    }
    __syncthreads();
    return v;  // valid in warp 0
}

// Part 2: channel-coupling terms.  grid (nb, ceil(nrhs/QT)); thread = channel c (strided), mesh point i = blockIdx.x.
//   r[(c,i),q] = acc[(c,i),q] - sum_{c' != c} V_cc'(r_i) X[(c',i),q]       (continues the double-double sum)
// V[i][c'][c] is read with c fastest (coalesced); X[(c',i),q] is staged in shared memory and broadcast.
// rmax (device double, pre-zeroed) receives max |r| (modulus).
__global__ void __launch_bounds__(RES_NT) resid_coupling_kernel(int nch, int nb, int nrhs, const double2 *__restrict__ V,
                                                               const double2 *__restrict__ X, long ldx,
                                                               double2 *__restrict__ R, const double2 *__restrict__ Rlo,
                                                               long ldr, double *rmax) {
    extern __shared__ __align__(16) unsigned char smraw[];
    double2 *Xs = reinterpret_cast<double2 *>(smraw);  // [QT][nch]
    __shared__ double shred[32];
    const int i = blockIdx.x, q0 = blockIdx.y * RES_QT;
    const int nq = min(RES_QT, nrhs - q0);
    for (int idx = threadIdx.x; idx < RES_QT * nch; idx += RES_NT) {
        const int qq = idx / nch, c2 = idx - qq * nch;
        Xs[idx] = qq < nq ? X[(long)(q0 + qq) * ldx + (long)c2 * nb + i] : make_double2(0.0, 0.0);
    }
    __syncthreads();
    double lmax = 0.0;
    const double2 *Vi = V + (long)i * nch * nch;
    for (int c = threadIdx.x; c < nch; c += RES_NT) {
        const long row = (long)c * nb + i;
        double sr[RES_QT], cr[RES_QT], si[RES_QT], ci[RES_QT];
#pragma unroll
        for (int qq = 0; qq < RES_QT; ++qq) {
            sr[qq] = si[qq] = cr[qq] = ci[qq] = 0.0;
            if (qq < nq) {
                const double2 h = R[(long)(q0 + qq) * ldr + row], l = Rlo[(long)(q0 + qq) * ldr + row];
                sr[qq] = h.x; si[qq] = h.y; cr[qq] = l.x; ci[qq] = l.y;
            }
        }
        for (int c2 = 0; c2 < nch; ++c2) {
            if (c2 == c) continue;
            const double2 v = Vi[(long)c2 * nch + c];
#pragma unroll
            for (int qq = 0; qq < RES_QT; ++qq) {
                const double2 x = Xs[qq * nch + c2];
                dd_mac(sr[qq], cr[qq], -v.x, x.x);
                dd_mac(sr[qq], cr[qq], v.y, x.y);
                dd_mac(si[qq], ci[qq], -v.x, x.y);
                dd_mac(si[qq], ci[qq], -v.y, x.x);
            }
        }
#pragma unroll
        for (int qq = 0; qq < RES_QT; ++qq)
            if (qq < nq) {
                const double re = __dadd_rn(sr[qq], cr[qq]), im = __dadd_rn(si[qq], ci[qq]);
                R[(long)(q0 + qq) * ldr + row] = make_double2(re, im);
                lmax = fmax(lmax, sqrt(re * re + im * im));
            }
    }
    lmax = block_max(lmax, shred);
    if (threadIdx.x == 0 && rmax) atomic_max_nonneg(rmax, lmax);
}

int structured_residual(cudaStream_t st, const StructTables &t, double energy, const double2 *V, int nrhs,
                        const double2 *Bx, long ldb, const double2 *X, long ldx, double2 *R, double2 *Rlo, long ldr,
                        double *rmax_dev) {
    if (nrhs <= 0) return 0;
    if (rmax_dev) HP_CUDA(cudaMemsetAsync(rmax_dev, 0, sizeof(double), st));
    {
        dim3 grid(t.nch, ceil_div(nrhs, RES_QT));
        const size_t smem = sizeof(double2) * RES_QT * t.nb;
        static SmemCfg cfg1;
        if (smem > 48 * 1024) HP_TRY(configure_smem(cfg1, resid_channel_kernel, smem));
        resid_channel_kernel<<<grid, RES_NT, smem, st>>>(t.nch, t.nb, nrhs, t.hT, t.dg0, t.ethr, energy, t.fa, V, Bx, ldb,
                                                         X, ldx, R, Rlo, ldr);
        HP_LAUNCHED();
    }
    {
        dim3 grid(t.nb, ceil_div(nrhs, RES_QT));
        const size_t smem = sizeof(double2) * RES_QT * t.nch;
        static SmemCfg cfg2;
        if (smem > 48 * 1024) HP_TRY(configure_smem(cfg2, resid_coupling_kernel, smem));
        resid_coupling_kernel<<<grid, RES_NT, smem, st>>>(t.nch, t.nb, nrhs, V, X, ldx, R, Rlo, ldr, rmax_dev);
        HP_LAUNCHED();
    }
    return 0;
}

// ---- the coupling part on the FP64 tensor cores ---------------------------------------------------------------------------
// The within-channel part (entries up to ~1e9: the end-point kinetic diagonal) is where the residual cancels and needs the
// double-double sum; the couplings are <= a few MeV, so sum_{c' != c} V_cc'(r_i) X[(c',i),q] in plain FP64 (DMMA) is exact
// to ~Nc 2^-53 |V_cc'| |X| ~ 1e-14 |X|, eight orders below |C||X|.  Per mesh point i that is one Nc x Nc by Nc x nrhs
// product: V_i (zero diagonal) times the point-major copy of X.  8 Nb Nc^3 flops at the DMMA rate instead of ~20x that many
// FP64 CUDA-core operations of the double-double loop (4.2 ms -> 0.5 ms per residual at cfg 3).
__global__ void __launch_bounds__(256) zero_diag_copy_kernel(int nch, long tot, const double2 *__restrict__ V,
                                                             double2 *__restrict__ Voff) {
    for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const int c1 = (int)(idx % nch), c2 = (int)((idx / nch) % nch);
        Voff[idx] = c1 == c2 ? make_double2(0.0, 0.0) : V[idx];
    }
}
int coupling_without_diagonal(cudaStream_t st, const StructTables &t, const double2 *V, double2 *Voff) {
    const long tot = (long)t.nb * t.nch * t.nch;
    zero_diag_copy_kernel<<<(int)std::min<long>(ceil_div(tot, 256), 148L * 16), 256, 0, st>>>(t.nch, tot, V, Voff);
    HP_LAUNCHED();
    return 0;
}

// Xp[(i nrhs + q) nch + c] = X[q ldx + c nb + i]: 32 x 32 tiles over (c, i), one right-hand side per blockIdx.z
__global__ void __launch_bounds__(256) to_point_major_kernel(int nch, int nb, int nrhs, const double2 *__restrict__ X, long ldx,
                                                             double2 *__restrict__ Xp) {
    __shared__ double2 tile[32][33];
    const int q = blockIdx.z, c0 = blockIdx.y * 32, i0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int k = ty; k < 32; k += 8) {  // read: i fastest
        const int c = c0 + k, i = i0 + tx;
        if (c < nch && i < nb) tile[k][tx] = X[(long)q * ldx + (long)c * nb + i];
    }
    __syncthreads();
    for (int k = ty; k < 32; k += 8) {  // write: c fastest
        const int i = i0 + k, c = c0 + tx;
        if (c < nch && i < nb) Xp[((long)i * nrhs + q) * nch + c] = tile[tx][k];
    }
}

// R[(c,i),q] = (hi + lo)[(c,i),q] - P[(i nrhs + q) nch + c]  (P == nullptr: no coupling term); rmax as above
__global__ void __launch_bounds__(256) resid_combine_kernel(int nch, int nb, int nrhs, double2 *__restrict__ R,
                                                            const double2 *__restrict__ Rlo, long ldr,
                                                            const double2 *__restrict__ P, double *rmax) {
    __shared__ double2 tile[32][33];
    __shared__ double shred[32];
    const int q = blockIdx.z, c0 = blockIdx.y * 32, i0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    if (P) {
        for (int k = ty; k < 32; k += 8) {  // read: c fastest
            const int i = i0 + k, c = c0 + tx;
            if (c < nch && i < nb) tile[tx][k] = P[((long)i * nrhs + q) * nch + c];
        }
        __syncthreads();
    }
    double lmax = 0.0;
    for (int k = ty; k < 32; k += 8) {  // i fastest
        const int c = c0 + k, i = i0 + tx;
        if (c < nch && i < nb) {
            const long at = (long)q * ldr + (long)c * nb + i;
            double2 h = R[at];
            const double2 l = Rlo[at];
            if (P) {
                const double2 p = tile[k][tx];
                // TwoSum of hi - p, the error joins the low word
                const double sr = __dsub_rn(h.x, p.x), br = __dsub_rn(sr, h.x);
                const double er = __dadd_rn(__dsub_rn(h.x, __dsub_rn(sr, br)), __dsub_rn(-p.x, br));
                const double si = __dsub_rn(h.y, p.y), bi = __dsub_rn(si, h.y);
                const double ei = __dadd_rn(__dsub_rn(h.y, __dsub_rn(si, bi)), __dsub_rn(-p.y, bi));
                h = make_double2(__dadd_rn(sr, __dadd_rn(l.x, er)), __dadd_rn(si, __dadd_rn(l.y, ei)));
            } else {
                h = make_double2(__dadd_rn(h.x, l.x), __dadd_rn(h.y, l.y));
            }
            R[at] = h;
            lmax = fmax(lmax, sqrt(h.x * h.x + h.y * h.y));
        }
    }
    lmax = block_max(lmax, shred);
    if (threadIdx.x == 0 && rmax) atomic_max_nonneg(rmax, lmax);
}

int zgemm_batched(cudaStream_t st, int m, int n, int k, double alpha, const double2 *A, long lda, long strideA,
                  const double2 *B, long ldb, long strideB, double beta, double2 *C, long ldc, long strideC, int nbatch);

int structured_residual_tc(cudaStream_t st, const StructTables &t, double energy, const double2 *V, const double2 *Voff,
                           const double2 *X, long ldx, double2 *R, double2 *Rlo, long ldr, double2 *Xp, double2 *Pp,
                           double *rmax_dev) {
    const int nrhs = t.nch;
    if (rmax_dev) HP_CUDA(cudaMemsetAsync(rmax_dev, 0, sizeof(double), st));
    {
        dim3 grid(t.nch, ceil_div(nrhs, RES_QT));
        const size_t smem = sizeof(double2) * RES_QT * t.nb;
        static SmemCfg cfg1;
        if (smem > 48 * 1024) HP_TRY(configure_smem(cfg1, resid_channel_kernel, smem));
        resid_channel_kernel<<<grid, RES_NT, smem, st>>>(t.nch, t.nb, nrhs, t.hT, t.dg0, t.ethr, energy, t.fa, V, nullptr, 0, X, ldx,
                                                         R, Rlo, ldr);
        HP_LAUNCHED();
    }
    const dim3 tgrid(ceil_div(t.nb, 32), ceil_div(t.nch, 32), nrhs);
    if (Voff) {
        to_point_major_kernel<<<tgrid, 256, 0, st>>>(t.nch, t.nb, nrhs, X, ldx, Xp);
        HP_LAUNCHED();
        HP_TRY(zgemm_batched(st, t.nch, nrhs, t.nch, 1.0, Voff, t.nch, (long)t.nch * t.nch, Xp, t.nch, (long)t.nch * nrhs, 0.0, Pp,
                             t.nch, (long)t.nch * nrhs, t.nb));
    }
    resid_combine_kernel<<<tgrid, 256, 0, st>>>(t.nch, t.nb, nrhs, R, Rlo, ldr, Voff ? Pp : nullptr, rmax_dev);
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- update + norms
// X += D; norms[0] = max|D|, norms[1] = max|X_new|  (moduli; norms pre-zeroed by the caller)
__global__ void __launch_bounds__(256) axpy_norm_kernel(long rows, int cols, double2 *__restrict__ X, long ldx,
                                                        const double2 *__restrict__ D, long ldd, double *norms,
                                                        const int *gate) {
    __shared__ double shred[32];
    if (gate != nullptr && *gate != 0) return;  // the refinement has already stopped: this step must not touch X
    double md = 0.0, mx = 0.0;
    const long tot = rows * cols;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long q = idx / rows, r = idx - q * rows;
        const double2 d = D[q * ldd + r];
        double2 x = X[q * ldx + r];
        x.x += d.x;
        x.y += d.y;
        X[q * ldx + r] = x;
        md = fmax(md, sqrt(d.x * d.x + d.y * d.y));
        mx = fmax(mx, sqrt(x.x * x.x + x.y * x.y));
    }
    md = block_max(md, shred);
    mx = block_max(mx, shred);
    if (threadIdx.x == 0) {
        atomic_max_nonneg(norms, md);
        atomic_max_nonneg(norms + 1, mx);
    }
}

int axpy_norm(cudaStream_t st, long rows, int cols, double2 *X, long ldx, const double2 *D, long ldd, double *norms_dev,
              const int *gate_dev) {
    HP_CUDA(cudaMemsetAsync(norms_dev, 0, 2 * sizeof(double), st));
    const long tot = rows * cols;
    if (tot <= 0) return 0;
    const int grid = (int)std::min<long>(ceil_div(tot, 256), 148L * 8);
    axpy_norm_kernel<<<grid, 256, 0, st>>>(rows, cols, X, ldx, D, ldd, norms_dev, gate_dev);
    HP_LAUNCHED();
    return 0;
}

// max modulus of a rows x cols block -> out[0] (pre-zeroed here)
__global__ void __launch_bounds__(256) maxabs_kernel(long rows, int cols, const double2 *__restrict__ X, long ldx, double *out) {
    __shared__ double shred[32];
    double mx = 0.0;
    const long tot = rows * cols;
    for (long idx = (long)blockIdx.x * blockDim.x + threadIdx.x; idx < tot; idx += (long)gridDim.x * blockDim.x) {
        const long q = idx / rows, r = idx - q * rows;
        const double2 x = X[q * ldx + r];
        mx = fmax(mx, sqrt(x.x * x.x + x.y * x.y));
    }
    mx = block_max(mx, shred);
    if (threadIdx.x == 0) atomic_max_nonneg(out, mx);
}

int maxabs(cudaStream_t st, long rows, int cols, const double2 *X, long ldx, double *out_dev) {
    HP_CUDA(cudaMemsetAsync(out_dev, 0, sizeof(double), st));
    const long tot = rows * cols;
    if (tot <= 0) return 0;
    const int grid = (int)std::min<long>(ceil_div(tot, 256), 148L * 8);
    maxabs_kernel<<<grid, 256, 0, st>>>(rows, cols, X, ldx, out_dev);
    HP_LAUNCHED();
    return 0;
}

__global__ void __launch_bounds__(256) maxabs_real_kernel(long n, const double *__restrict__ x, double *out) {
    __shared__ double shred[32];
    double m = 0.0;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) m = fmax(m, fabs(x[i]));
    m = block_max(m, shred);
    if (threadIdx.x == 0) atomic_max_nonneg(out, m);
}

// out (pre-zeroed by the caller) <- max(out, max_i |x_i|)
int maxabs_real(cudaStream_t st, long n, const double *x, double *out_dev) {
    if (n <= 0) return 0;
    const int grid = (int)std::min<long>(ceil_div(n, 256), 148L * 8);
    maxabs_real_kernel<<<grid, 256, 0, st>>>(n, x, out_dev);
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- backward error
// out[0] = max_q  ||r_q||_inf / (anorm * ||x_q||_inf + ||b_q||_inf)   (one CTA per right-hand side; out pre-zeroed)
__global__ void __launch_bounds__(256) backward_err_kernel(long rows, const double2 *__restrict__ R, long ldr,
                                                           const double2 *__restrict__ X, long ldx,
                                                           const double *__restrict__ anorm_p,
                                                           const double *__restrict__ bnorm_p, double *out) {
    __shared__ double shred[32];
    const long q = blockIdx.x;
    double mr = 0.0, mx = 0.0;
    for (long r = threadIdx.x; r < rows; r += blockDim.x) {
        const double2 a = R[q * ldr + r], x = X[q * ldx + r];
        mr = fmax(mr, sqrt(a.x * a.x + a.y * a.y));
        mx = fmax(mx, sqrt(x.x * x.x + x.y * x.y));
    }
    mr = block_max(mr, shred);
    mx = block_max(mx, shred);
    if (threadIdx.x == 0) {
        const double den = *anorm_p * mx + *bnorm_p;
        atomic_max_nonneg(out, den > 0.0 ? mr / den : 0.0);
    }
}

int backward_error(cudaStream_t st, long rows, int nrhs, const double2 *R, long ldr, const double2 *X, long ldx,
                   const double *anorm_dev, const double *bnorm_dev, double *out_dev) {
    HP_CUDA(cudaMemsetAsync(out_dev, 0, sizeof(double), st));
    if (nrhs <= 0) return 0;
    backward_err_kernel<<<nrhs, 256, 0, st>>>(rows, R, ldr, X, ldx, anorm_dev, bnorm_dev, out_dev);
    HP_LAUNCHED();
    return 0;
}

// ||C - E I||_inf from the block structure: row (c,i): sum_j |hT_ij| (j != i) + |Cdiag| + sum_{c' != c} |V_cc'(r_i)|
__global__ void __launch_bounds__(256) anorm_kernel(int nch, int nb, const double *__restrict__ hT,
                                                    const double *__restrict__ dg0, const double *__restrict__ ethr,
                                                    double energy, const double2 *__restrict__ V, double *out) {
    __shared__ double shred[32];
    const int N = nch * nb;
    double best = 0.0;
    for (int row = blockIdx.x * blockDim.x + threadIdx.x; row < N; row += gridDim.x * blockDim.x) {
        const int c = row / nb, i = row - c * nb;
        double s = 0.0;
        for (int j = 0; j < nb; ++j)
            if (j != i) s += fabs(hT[(long)j * nb + i]);
        for (int c2 = 0; c2 < nch; ++c2) {
            const double2 v = V[((long)i * nch + c2) * nch + c];
            if (c2 == c) {
                const double dr = __dadd_rn(__dadd_rn(dg0[row], __dsub_rn(ethr[c], energy)), v.x);
                s += sqrt(dr * dr + v.y * v.y);
            } else {
                s += sqrt(v.x * v.x + v.y * v.y);
            }
        }
        best = fmax(best, s);
    }
    best = block_max(best, shred);
    if (threadIdx.x == 0) atomic_max_nonneg(out, best);
}

int structured_anorm(cudaStream_t st, const StructTables &t, double energy, const double2 *V, double *out_dev) {
    HP_CUDA(cudaMemsetAsync(out_dev, 0, sizeof(double), st));
    const int N = t.nch * t.nb;
    anorm_kernel<<<ceil_div(N, 256), 256, 0, st>>>(t.nch, t.nb, t.hT, t.dg0, t.ethr, energy, V, out_dev);
    HP_LAUNCHED();
    return 0;
}

// ---------------------------------------------------------------------------------------------------- contraction
// R[c1,c2] = (h2m/a) sum_i fa_i X[(c1,i), c2]  -- one warp per output element, plain transpose (no conjugate).
__global__ void __launch_bounds__(256) contract_kernel(int nch, int nb, double pref, const double *__restrict__ fa,
                                                       const double2 *__restrict__ X, long ldx, double2 *__restrict__ R) {
    const long w = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= (long)nch * nch) return;
    const int c2 = (int)(w / nch), c1 = (int)(w - (long)c2 * nch);
    const double2 *x = X + (long)c2 * ldx + (long)c1 * nb;
    double sr = 0.0, si = 0.0;
    for (int i = lane; i < nb; i += 32) {
        const double f = fa[i];
        const double2 v = x[i];
        sr = fma(f, v.x, sr);
        si = fma(f, v.y, si);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sr += __shfl_xor_sync(0xffffffffu, sr, off);
        si += __shfl_xor_sync(0xffffffffu, si, off);
    }
    if (lane == 0) R[(long)c2 * nch + c1] = make_double2(pref * sr, pref * si);
}

int contract_with(cudaStream_t st, const StructTables &t, const double *fa_dev, const double2 *X, long ldx, double2 *R) {
    const long warps = (long)t.nch * t.nch;
    contract_kernel<<<ceil_div(warps * 32, 256), 256, 0, st>>>(t.nch, t.nb, t.h2m / t.a, fa_dev, X, ldx, R);
    HP_LAUNCHED();
    return 0;
}

int contract(cudaStream_t st, const StructTables &t, const double2 *X, long ldx, double2 *R) {
    const long warps = (long)t.nch * t.nch;
    contract_kernel<<<ceil_div(warps * 32, 256), 256, 0, st>>>(t.nch, t.nb, t.h2m / t.a, t.fa, X, ldx, R);
    HP_LAUNCHED();
    return 0;
}

}  // namespace hp
