/* tdde_bench.h -- measurement helpers, test exports and the same-box comparator of libtdde.so.  None of these is on the product
 * path (tdde.h); they are compiled into the library only with -DTDDE_WITH_BENCH (paper_2512_21697_b200/build.py sets it; a
 * production build can leave it out) and are what bench.py and tests/ call. */
#ifndef TDDE_BENCH_H_
#define TDDE_BENCH_H_

#include "tdde.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Pin P11 support: one CN step that runs exactly n_iters full BiCGSTAB iterations with every exit test
 * disabled.  trace_dev (device, nullable): [n_iters][8][n] complex128 receiving, after each iteration, the
 * vectors p, v, s, t, x, r, y, z (this order, boundary layout).  Synchronises. */
int tdde_step_forced(tdde_handle* h, tdde_c64* c_dev, const double* g_mid, int32_t n_iters, tdde_c64* trace_dev);

/* Test export of the kernel an iteration uses for v = A y on the banded path (R21): y = addv + beta sum_L g[L] (A_L (x) R_L) x
 * with the fused sums dots[0..1] = <aux, y> (re, im), dots[2] = ||y||^2 over all n elements (aux_dev nullable: dots[0..1] = 0).
 * which: 0 = the kernel the handle would use (DMMA variant when the shape has one), 1 = force the register-window kernel.
 * x_dev, addv_dev, aux_dev, y_dev: device, n complex128, boundary layout, y must not alias the inputs; dots: host [3], nullable.
 * TDDE_EINVAL when the handle is not on the banded path (tdde_apply_path != 1) or has no terms.  Synchronises. */
int tdde_apply_coupling(tdde_handle* h, tdde_c64 beta, const double* g, const tdde_c64* x_dev, const tdde_c64* addv_dev,
                        const tdde_c64* aux_dev, tdde_c64* y_dev, int32_t which, double* dots);

/* Measurement helpers (timed in bench.py; no effect on state).
 *   tdde_time_kernel: enqueue `reps` launches of one internal kernel on the handle's stream between two CUDA
 *   events and return the mean milliseconds per launch in *ms_out.  which: 0 = operator apply v = A y with
 *   fused <rhat,v>; 1 = preconditioner apply; 2 = p-update; 3 = s-update; 4 = x,r-update; 5 = boundary<->internal
 *   transpose; 6 = S-only apply (norm).  g: host [n_terms] used by which == 0.  Synchronises.
 *   tdde_fp64_peak: run an unrolled independent-DFMA kernel on every SM and return achieved FLOP/s. */
int tdde_time_kernel(tdde_handle* h, int32_t which, int32_t reps, const double* g, double* ms_out);
int tdde_fp64_peak(void* cuda_stream, double* flops_out);
/* The same for the pipe k_apply_mma runs on: mode 0 = DFMA only, 1 = DMMA only (mma.sync.m8n8k4.f64), 2 = 8 DMMA : 32 DFMA mixed in one warp.
 * On B200 all three land on one peak (DMMA and DFMA share the FP64 pipe), the mix about 12 % below it. */
int tdde_fp64_pipe_probe(void* cuda_stream, int32_t mode, double* flops_out);

/* Comparator, not on the product path: the paper's own formulation on this GPU.  Allocates the global
 * CSR matrix A = S + i dt/2 H(g) (structure once), recomputes every non-zero from the stored radial and
 * angular matrices with one assembly kernel and forms y = A x by CSR SpMV, `reps` times
 * each; mean milliseconds go to *ms_assemble / *ms_spmv (host, nullable), the non-zero count to *nnz (host, nullable).
 * x_dev, y_dev: device, n complex128, boundary layout, must not alias.  Needs 20 bytes of device memory per non-zero.
 * Only for problems on the banded apply path (tdde_apply_path == 1), else TDDE_EINVAL.  Synchronises. */
int tdde_paper_variant(tdde_handle* h, const double* g, const tdde_c64* x_dev, tdde_c64* y_dev, int32_t reps,
                       double* ms_assemble, double* ms_spmv, int64_t* nnz);

/* Host-only self-test of the set-up code behind tdde_precond (no GPU needed): builds a random banded
 * M = S + i tau H of size n and half-bandwidth w, the partitioned factors for P partitions, replays the
 * solve on the host and writes the relative residual ||M y - b|| / ||b|| to *rel_res (host).  Returns the number of
 * partitions actually used (>= 1; the plan shrinks P until interiors are >= 8 w rows) or a negative tdde_status. */
int tdde_selftest_partition(int32_t n, int32_t w, int32_t P, uint32_t seed, double* rel_res);

/* Which kernel an iteration uses for v = A y: 0 = k_apply_generic, 1 = k_apply_banded (register window), 2 = k_apply_sparse (staged),
 * 3 = k_apply_mma (banded path, radial contraction on the FP64 tensor-core path). */
int tdde_iter_apply_kernel(const tdde_handle* h);

/* Host-only self-test of the operand table behind k_apply_mma (no GPU needed): random column bands R_L of half-bandwidth w (3, 6 or 9)
 * and size n_rad, T terms; builds the MMA fragment table, replays the kernel's slice / tile / three-product arithmetic on the host for
 * one channel and writes max_i |y_i - sum_L (R_L z_L)_i| / max_i |.| to *max_rel_err (host). */
int tdde_selftest_mma_frags(int32_t n_rad, int32_t w, int32_t T, uint32_t seed, double* max_rel_err);

/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
int64_t tdde_launch_count(const tdde_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* TDDE_BENCH_H_ */
