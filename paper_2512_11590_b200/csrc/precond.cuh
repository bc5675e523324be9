// precond.cuh -- FP64 block-diagonal preconditioner and precision moves of the mixed path (precond.cu).
#pragma once
#include "structured.cuh"

namespace hp {

// Kinv[c] <- K_c^-1, K_c = diagonal block c of C - E*I (nb x nb complex128, column-major, blocks contiguous).
// info_dev (pre-zeroed by the caller) receives c*nb + k + 1 if block c has no non-zero pivot at step k.
// W != nullptr (non-local potentials): K_c = kinetic/diagonal terms + the full diagonal block (c,c) of the N x N matrix W
int precond_invert(cudaStream_t st, const StructTables &t, double energy, const double2 *V, double2 *Kinv, int *info_dev,
                   const double2 *W = nullptr, long ldw = 0);
// S <- K_d^-1 (C - E*I) in split complex64 (identity diagonal blocks, Kinv_c * diag V_cc' elsewhere)
int precond_assemble(cudaStream_t st, const StructTables &t, const double2 *Kinv, const double2 *V, CView S);
// non-local potentials: S <- K_d^-1 (C - E*I) with full blocks of W; T: N x nch complex128 scratch (ld ldt)
int precond_assemble_nonlocal(cudaStream_t st, const StructTables &t, const double2 *Kinv, const double2 *W, long ldw, CView S,
                              double2 *T, long ldt);
// the same two in complex128 (preconditioned FP64 factorisation)
int precond_assemble_z(cudaStream_t st, const StructTables &t, const double2 *Kinv, const double2 *V, ZView S);
int precond_rhs_z(cudaStream_t st, const StructTables &t, const double2 *Kinv, ZView B);
// B <- K_d^-1 * (surface right-hand sides), split complex64, N x nch
int precond_rhs(cudaStream_t st, const StructTables &t, const double2 *Kinv, CView B);
// D <- (complex64) Z
int demote(cudaStream_t st, long rows, int cols, const double2 *Z, long ldz, CView D);
// X <- (accumulate ? X : 0) + D;  norms_dev[0] = max|D|, norms_dev[1] = max|X|.  gate_dev (device int, may be nullptr):
// when it reads non-zero the kernel does nothing (norms stay zero) -- a refinement step enqueued after the device-side
// stopping rule has fired
int promote_add(cudaStream_t st, long rows, int cols, double2 *X, long ldx, CView D, bool accumulate, double *norms_dev,
                const int *gate_dev = nullptr);

// The paper's Type 3 in its literal form (Eqs. 7-9): point-major Schur matrix S = I + K^-1 V with K the real
// kinetic block shared by all channels.  KTinv: nb x nb column-major inverse of h2m*T; cf: [nch*nb] centrifugal terms
// h2m l(l+1)/r_i^2; g = KTinv q2 (nb).  All three are energy-independent (computed once at setup).
int type3_assemble(cudaStream_t st, const StructTables &t, const double *KTinv, const double *cf, double energy, const double2 *V,
                   CView S);
int type3_rhs(cudaStream_t st, const StructTables &t, const double *g, CView B);
// X (channel-major complex128) <- point-major complex64 solution; norms_dev[1] = max|X|
int type3_promote(cudaStream_t st, const StructTables &t, CView Xs, double2 *X, long ldx, double *norms_dev);

}  // namespace hp
