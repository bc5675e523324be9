/*
 * hprmat_profile.h -- measurement aids of bench.py; NOT part of the product interface (include/hprmat.h).
 *
 * libhprmat.so exports the per-launch timing record and the launch counter below; the FP64 tensor-core peak probe lives
 * in a library of its own (libhprmat_bench.so, built from paper_2512_11590_b200/bench_csrc/) that the product never loads.
 */
#ifndef HPRMAT_PROFILE_H
#define HPRMAT_PROFILE_H

#ifdef __cplusplus
extern "C" {
#endif

/* While enabled, every launch of the GEMM, panel, row-interchange and inverse kernels inside the LU and the triangular
 * solves is bracketed by a CUDA-event pair on its stream (which also serialises the side stream's work into the sums, and
 * switches the CUDA-graph replay of the factorisation off).  Process-wide record; hprmat_profile_read synchronises those
 * events, returns the summed GEMM milliseconds, the summed algorithmic flops (8 m n k per launch) and the launch count, and
 * resets the record. */
int hprmat_profile(int enable);
int hprmat_profile_read(double *ms, double *flops, long long *launches);
/* Per-category totals of the record consumed by the last hprmat_profile_read: cat 0 = trailing-update GEMMs of the LU,
 * 1 = GEMMs of the U12 triangular solves inside the LU, 2 = panel factorisations (top-block kernel, L21 product and its
 * check; or the pivoting panel kernels), 3 = row interchanges, 4 = GEMMs of the right-hand-side triangular solves,
 * 5 = other.  ms/flops/launches host, may be NULL. */
int hprmat_profile_cat(int cat, double *ms, double *flops, long long *launches);
/* number of kernel launches issued by libhprmat.so since process start, kernels replayed from a CUDA graph included
 * (bench.py's gpu_launches) */
long long hprmat_launch_count(void);

/* Which tcgen05 kernel serves the planar complex64 GEMM (hprmat_cgemm_tf32 and every such product inside the mixed modes):
 * 0 = automatic (default: the persistent kernel, CTA pairs / cta_group::2 when there is more than one 128-row tile),
 * 1 = the one-tile-per-CTA kernel (cgemm.cu), 2 = persistent single CTAs, 3 / 4 = persistent CTA pairs with 256 x 128 /
 * 256 x 256 tiles, 5 = as 0 but the cluster split-K kernel (cgemm_splitk.cu) wherever its preconditions hold.  Any other
 * value only queries.  Returns the setting in force.  Process-wide; for A/B measurements. */
int hprmat_profile_cgemm_variant(int variant);

/* Which kernel serves the FP32-class ("3xTF32") planar complex64 GEMM (hprmat_cgemm_3xtf32 and the products of the
 * escalated factorisations): 0 = automatic (tcgen05 with the lo parts computed in shared memory, cgemm3x.cu, when C is
 * distinct from A and B and the problem fills >= 32 tiles; else the mma.sync kernel, cgemm3.cu), 1 = mma.sync always,
 * 2 = tcgen05 whenever legal.  Returns 0, or -1 for another value.  Process-wide; for tests and A/B measurements. */
int hprmat_profile_cgemm3_variant(int variant);

/* Programmatic dependent launch of the small kernels of the complex64 LU (their prologues overlap the predecessor's tail):
 * 1 = on (default), 0 = off, any other value only queries.  Returns the setting in force.  Process-wide; A/B measurements. */
int hprmat_profile_pdl(int enable);

/* Look-ahead inside the factorisations with verified diagonal pivots (the update of the columns the next panel does not need yet
 * runs on another stream, under that panel's factorisation): 1 = on (default), 0 = off, any other value only queries.
 * Returns the setting in force.  Process-wide; A/B measurements. */
int hprmat_profile_lookahead(int enable);

/* How many launch sequences (factorisations, triangular solves) of the context are replayed from CUDA graphs (captured) and
 * how many had to stay plain stream launches (eager: capture refused).  captured / eager: host, may be NULL. */
struct hprmat_ctx;
int hprmat_profile_graphs(const struct hprmat_ctx *ctx, int *captured, int *eager);

/* libhprmat_bench.so: FP64 tensor-core (DMMA, mma.sync.m8n8k4.f64) issue-rate ceiling of the device, measured with a
 * register-resident loop (no memory traffic) on 148*ctas_per_sm CTAs of 8 warps, `iters` x 8 MMAs per warp.
 * tflops (host, out): real TFLOP/s; ms (host, out, may be NULL): device time of the timed launch.  Synchronises. */
int hprmat_bench_dmma_peak(void *cuda_stream, int iters, int ctas_per_sm, double *tflops, double *ms);

#ifdef __cplusplus
}
#endif
#endif /* HPRMAT_PROFILE_H */
