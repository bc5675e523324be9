// structured.cuh -- device tables of the Lagrange-Legendre problem and the O(N^2) kernels around the LU.
#pragma once
#include <algorithm>

#include "common.cuh"

namespace hp {

// Device-resident tables computed once at hprmat_setup.
struct StructTables {
    int nch = 0, nb = 0;
    double a = 0, h2m = 0;
    const double *hT = nullptr;    // nb x nb column-major: (double)(h2m * T_ij), T = kinetic + Bloch in units h2m = 1
    const double *dg0 = nullptr;   // [nch*nb]: h2m*T_ii + h2m*l_c(l_c+1)/r_i^2
    const double *ethr = nullptr;  // [nch]
    const double *fa = nullptr;    // [nb]: f_i(a)
};

int assemble_z(cudaStream_t st, const StructTables &t, double energy, const double2 *V, double2 *C, long ldc);
// non-local potentials: C <- W + (kinetic + Bloch + centrifugal + threshold - E on the diagonal blocks); W N x N, ld ldw
int assemble_nonlocal(cudaStream_t st, const StructTables &t, double energy, const double2 *W, long ldw, double2 *C, long ldc);
// out_dev <- ||W + diagonal-block terms||_inf; rowsum_scratch: N doubles
int nonlocal_anorm(cudaStream_t st, const StructTables &t, double energy, const double2 *W, long ldw, double *rowsum_scratch,
                   double *out_dev);
int maxabs_real(cudaStream_t st, long n, const double *x, double *out_dev);
int build_rhs(cudaStream_t st, const StructTables &t, double2 *B, long ldb);
// R <- Bx - (C - E I) X (Bx == nullptr: the surface right-hand sides), double-double accumulation; Rlo is scratch of
// the same shape as R; rmax_dev (may be nullptr) receives max |R_ij|.
int structured_residual(cudaStream_t st, const StructTables &t, double energy, const double2 *V, int nrhs,
                        const double2 *Bx, long ldb, const double2 *X, long ldx, double2 *R, double2 *Rlo, long ldr,
                        double *rmax_dev);
// X += D; norms_dev[0] = max|D|, norms_dev[1] = max|X|.  gate_dev: as in promote_add (precond.cuh)
// Voff <- V with the channel-diagonal entries V_cc(r_i) zeroed (they belong to the within-channel, double-double part)
int coupling_without_diagonal(cudaStream_t st, const StructTables &t, const double2 *V, double2 *Voff);
// Same residual for the nch surface right-hand sides, the coupling part as one batched DMMA product per mesh point on the
// point-major copy of X (within-channel part still double-double).  Voff == nullptr: no coupling term (V = 0).
// Xp, Pp: N x nch scratch each.
int structured_residual_tc(cudaStream_t st, const StructTables &t, double energy, const double2 *V, const double2 *Voff,
                           const double2 *X, long ldx, double2 *R, double2 *Rlo, long ldr, double2 *Xp, double2 *Pp,
                           double *rmax_dev);
int axpy_norm(cudaStream_t st, long rows, int cols, double2 *X, long ldx, const double2 *D, long ldd, double *norms_dev,
              const int *gate_dev = nullptr);
int maxabs(cudaStream_t st, long rows, int cols, const double2 *X, long ldx, double *out_dev);
// out_dev <- max_q ||r_q||_inf / (anorm ||x_q||_inf + bnorm); anorm and bnorm are read from DEVICE memory, so that the whole
// report can be enqueued without a host round trip
int backward_error(cudaStream_t st, long rows, int nrhs, const double2 *R, long ldr, const double2 *X, long ldx,
                   const double *anorm_dev, const double *bnorm_dev, double *out_dev);
int structured_anorm(cudaStream_t st, const StructTables &t, double energy, const double2 *V, double *out_dev);
int contract(cudaStream_t st, const StructTables &t, const double2 *X, long ldx, double2 *R);
// same with another surface vector (sector matrices of the propagation: left / right end)
int contract_with(cudaStream_t st, const StructTables &t, const double *fa_dev, const double2 *X, long ldx, double2 *R);

}  // namespace hp
