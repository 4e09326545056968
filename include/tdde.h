/* tdde.h -- C ABI of the B200 Crank-Nicolson / BiCGSTAB Dirac propagator (libtdde.so).
 *
 * One thing is computed: the implicit Crank-Nicolson step of the time-dependent Dirac equation in a
 * (kappa,mu) x radial-B-spline basis (Eq. 25, with H at the midpoint of PAPER.md:195, Eq. 22)
 *
 *     (S + i dt/2 H(t_{n+1/2})) c^{n+1} = (S - i dt/2 H(t_{n+1/2})) c^n ,
 *     H(t) = H0 + sum_L g_L(t) (A_L (x) R_L)                     (block form: Eq. 17)
 *
 * solved by BiCGSTAB preconditioned with M = S + i dt/2 H0 (Eq. 26),
 * which is block-diagonal over angular channels and is applied through per-class
 * banded LU factors.  The assembled matrix H(t) is never stored.
 *
 * Conventions (all entry points):
 *   - "host" / "device" is stated per pointer.  Device pointers are plain CUDA device addresses
 *     (e.g. torch.Tensor.data_ptr()), 16-byte aligned; the library neither frees nor keeps them.
 *   - state vectors: c[a * n_rad + j], a = angular channel (one (kappa,mu) pair), j = radial index over
 *     both components, complex128 interleaved (re, im), contiguous, length n = n_ang * n_rad.
 *   - a radial band matrix R of half-bandwidth w: row-major band[i][d + w] = R[i][i + d], -w <= d <= w,
 *     entries with i + d outside [0, n_rad) are ignored.
 *   - every call returns 0 on success or a negative tdde_status; nothing throws or aborts across the ABI.
 *   - all device work is enqueued on the CUDA stream given to tdde_create.
 *   - there is no CPU fallback: every call fails with TDDE_ECUDA when no CUDA device is usable.
 *   - a handle belongs to the device that was current at tdde_create; every call runs there whatever the caller's current device.
 * Measurement helpers, test exports and the paper-variant comparator are declared in tdde_bench.h (compiled in with -DTDDE_WITH_BENCH).
 */
#ifndef TDDE_H_
#define TDDE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tdde_handle tdde_handle;        /* opaque; owned by the library, freed by tdde_destroy */
typedef struct { double re, im; } tdde_c64;    /* == numpy complex128 */

typedef enum {
  TDDE_OK         =  0,
  TDDE_EINVAL     = -1,  /* null pointer, non-positive dims, w >= n_rad, CSR column out of range, bad rowptr, bad class */
  TDDE_ENOMEM     = -2,  /* host or device allocation failed */
  TDDE_ECUDA      = -3,  /* a CUDA runtime call failed; text via tdde_last_cuda_error() */
  TDDE_ESINGULAR  = -4,  /* zero / non-finite pivot in the banded LU of some M_k = S_k + i dt/2 H0_k */
  TDDE_EBREAKDOWN = -5,  /* |rho|, |<rhat,v>| or <t,t> below 1e-290 or non-finite (BiCGSTAB breakdown) */
  TDDE_ENOCONV    = -6   /* max_iter full iterations without reaching rtol */
} tdde_status;

typedef struct {
  int32_t n_ang;     /* angular channels (kappa,mu)                                  PAPER.md:94 (Eq. 7)   */
  int32_t n_rad;     /* 2*N_r: radial index over both components, interleaved                               */
  int32_t n_cls;     /* distinct field-free blocks (kappa-classes), 1..n_ang          */
  int32_t w0;        /* half-bandwidth of S_k and H0_k                                                      */
  int32_t n_terms;   /* T, number of coupling terms g_L (A_L (x) R_L); may be 0                             */
  int32_t max_iter;  /* full BiCGSTAB iterations per step before TDDE_ENOCONV                               */
  double  dt;        /* time step (a.u.); may be negative (time reversal)                                   */
  double  rtol;      /* stop when ||r||_2 <= rtol * ||b||_2                                                 */
} tdde_config;

typedef struct {               /* one coupling term g_L(t) * (A_L (x) R_L)      PAPER.md:155-163 (Eq. 17)   */
  int32_t w;                   /* half-bandwidth of R_L                                                     */
  int32_t reserved;            /* set to 0                                                                  */
  const tdde_c64* R_band;      /* host [n_rad][2w+1]                                                        */
  const int32_t*  A_rowptr;    /* host CSR of A_L, n_ang + 1 entries, non-decreasing, A_rowptr[0] = 0       */
  const int32_t*  A_col;       /* host [nnz], 0 <= col < n_ang                                              */
  const tdde_c64* A_val;       /* host [nnz]                                                                */
} tdde_term;

typedef struct {
  int64_t steps;        /* CN steps completed by the call                                                   */
  int64_t half_iters;   /* BiCGSTAB half-iterations summed over those steps (a full iteration counts 2;
                           the ||s|| exit leaves an odd count for its step)                                 */
  int64_t applies;      /* operator applies (A or B times a vector) enqueued and executed                   */
  int64_t preconds;     /* preconditioner applies executed                                                  */
  double  rel_res;      /* ||r|| / ||b|| at the exit of the last step                                       */
  int32_t status;       /* tdde_status of the last step                                                     */
  int32_t last_half_iters; /* half-iterations of the last step                                              */
} tdde_stats;

/* Build a propagator.  Copies every host input (caller may free them on return), forms per class
 * M+-_k = S_k +- i dt/2 H0_k, factorises M+_k = L U without pivoting (legitimate because the Hermitian part
 * of M+_k is S_k > 0), allocates ~10 work vectors of n complex128 on the current device.
 *   S_band, H0_band : host [n_cls][n_rad][2*w0+1]
 *   cls_of_chan     : host [n_ang], values in [0, n_cls)
 *   terms           : host [n_terms]
 *   cuda_stream     : cudaStream_t (as void*), 0 = legacy default stream
 * Errors: TDDE_EINVAL, TDDE_ENOMEM, TDDE_ECUDA, TDDE_ESINGULAR; *out is NULL on failure. */
int tdde_create(tdde_handle** out, const tdde_config* cfg, const tdde_c64* S_band, const tdde_c64* H0_band,
                const int32_t* cls_of_chan, const tdde_term* terms, void* cuda_stream);

/* One CN step in place on c_dev (device, n complex128).  g_mid: host [n_terms], g_L(t_{n+1/2}).
 * The call synchronises the stream once at its end (the speculative step driver must learn whether a step ran out
 * of enqueued iterations) and returns the step's status; *st (nullable) receives the statistics.  There is no host
 * synchronisation per BiCGSTAB iteration.  On failure c_dev holds the last iterate. */
int tdde_step(tdde_handle* h, tdde_c64* c_dev, const double* g_mid, tdde_stats* st);

/* n_steps CN steps in place on c_dev.  g_table: host [n_steps][n_terms], row s = g_L at the midpoint of step s.
 * Stops at the first failing step (st->steps tells how many completed).  Device state is read back once per batch
 * of 64 steps and once at the end; the call returns synchronised.  st is nullable. */
int tdde_propagate(tdde_handle* h, tdde_c64* c_dev, int64_t n_steps, const double* g_table, tdde_stats* st);

/* *out (host) = Re(c^H S c), the total probability in the non-orthogonal basis (S: PAPER.md:178-182).
 * Synchronises. */
int tdde_norm(tdde_handle* h, const tdde_c64* c_dev, double* out);

/* Test / measurement export: y = alpha S x + beta (H0 + sum_L g[L] A_L (x) R_L) x.
 * g: host [n_terms] (may be NULL when n_terms == 0).  x_dev, y_dev: device, n complex128, must not alias.
 * Does not synchronise. */
int tdde_apply(tdde_handle* h, tdde_c64 alpha, tdde_c64 beta, const double* g, const tdde_c64* x_dev,
               tdde_c64* y_dev);

/* Test / measurement export: y = (S + i dt/2 H0)^{-1} x, block-Jacobi over channels.
 * x_dev, y_dev: device, n complex128; may alias.  Does not synchronise. */
int tdde_precond(tdde_handle* h, const tdde_c64* x_dev, tdde_c64* y_dev);

/* Same as tdde_step / tdde_propagate but with HOST state vectors: c_host (n complex128) is copied to the
 * device, propagated and copied back; synchronises.  This is the end-to-end entry bench.py's "e2e" times. */
int tdde_propagate_host(tdde_handle* h, tdde_c64* c_host, int64_t n_steps, const double* g_table, tdde_stats* st);

/* Observables (Eq. 33: dP/dE = sum_{kappa,mu} |<psi_{kappa,mu,E}|Psi>|^2 with psi the field-free
 * eigenstates of PAPER.md:174-184, Eq. 19-20, which depend on kappa only).
 * tdde_set_eigenstates copies n_states eigenvectors per kappa-class to the device: V host [n_cls][n_states][n_rad], row e of class k =
 *   eigenvector e of the pencil (H0_k, S_k), normalised as the caller wants the probabilities normalised (v^H S_k v = 1 for
 *   probabilities), e.g. the output of tdde_eigensolve.
 * tdde_eigensolve (no handle needed): ALL eigenpairs of the n_cls Hermitian-definite pencils (H0_k, S_k) of PAPER.md Eq. 20 on the current
 *   device, batched over the classes (banded Cholesky of S_k, reduction to standard form, cyclic Jacobi with the round-robin parallel
 *   ordering, back-transformation).  S_band, H0_band: host [n_cls][n_rad][2*w0+1] as for tdde_create; E_host [n_cls][n_rad] ascending;
 *   V_host (nullable) [n_cls][n_rad][n_rad], row e = eigenvector of E[e], S-orthonormal -- the layout tdde_set_eigenstates takes.
 *   Set-up work (the paper solves these once, "2 kappa_max separate eigenvalue problems of dimension 2N"): dense O(n_rad^3) per class,
 *   n_rad <= 4096.  TDDE_ESINGULAR when some S_k is not positive definite.  Synchronises.
 * tdde_project: P_host [n_ang][n_states] receives |v_{k(a),e}^H S_k c_a|^2 for every channel a (the inner product of the
 *   non-orthogonal basis).  c_dev: device, n complex128.  Synchronises.  TDDE_EINVAL before tdde_set_eigenstates. */
int tdde_set_eigenstates(tdde_handle* h, int32_t n_states, const tdde_c64* V);
int tdde_project(tdde_handle* h, const tdde_c64* c_dev, double* P_host);
int tdde_eigensolve(int32_t n_cls, int32_t n_rad, int32_t w0, const tdde_c64* S_band, const tdde_c64* H0_band, double* E_host,
                    tdde_c64* V_host, void* cuda_stream);

/* ---- Channel-slab sharding over several GPUs (SURVEY 8(f) NEXT-3; PAPER.md:279-297 section 3.2, :307 section 3.3) ----
 * The paper partitions the angular channels among the ranks, exchanges the coupled x-slabs before every operator apply, keeps the
 * block-diagonal preconditioner rank-local and sums every inner product over the ranks.  Here: a SHARD is an ordinary handle created
 * from the rank-local problem (channels [halo | owned | halo] renumbered from 0, rows of every A_L for the owned channels only;
 * paper_2512_21697_b200/sharding.py builds it), a GROUP drives the shards of one process in lock step:
 *   before each apply the halo channels of its input vector are refreshed from their owners (device copies between local shards,
 *   pack + ncclSend/ncclRecv + unpack between ranks); every kernel writes and sums owned channels only; the three partial sums of a
 *   fused reduction are all-reduced (ncclAllReduce) between the kernel's block pass and the scalar update (k_finalize), everything
 *   stream-ordered; one host read of the solver state per CN step.
 * n_local = 1 with an NCCL id = one shard per process / GPU (production); n_local = world with nccl_id = NULL = every shard in this
 * process on one stream (how the exchange, the ownership masks and the split reductions are tested on a one-GPU box).
 *   own_lo, own_hi : owned channels [own_lo, own_hi) in the shard's LOCAL numbering
 *   recv_*         : halo pieces: channels [recv_lo, recv_lo + recv_n) of this shard = channels [recv_src_lo, ...) of shard recv_rank
 *   send_*         : the same pieces seen from the owner (needed with NCCL only): channels [send_lo, send_lo + send_n) go to send_rank
 * While a handle is attached to a group only tdde_group_propagate may drive it (its fused reductions hand their sums to the group);
 * tdde_group_destroy detaches it.  All shards must share n_rad, n_terms, dt, rtol, max_iter, the device and the stream.  Errors: TDDE_EINVAL, TDDE_ENOMEM, TDDE_ECUDA (also: NCCL not loadable). */
typedef struct tdde_group tdde_group;
typedef struct {
  int32_t rank, world;
  int32_t own_lo, own_hi;
  int32_t n_recv;
  const int32_t *recv_rank, *recv_lo, *recv_src_lo, *recv_n;   /* host [n_recv] */
  int32_t n_send;
  const int32_t *send_rank, *send_lo, *send_n;                 /* host [n_send] */
} tdde_shard;
int  tdde_nccl_unique_id(void* id128);                          /* host, 128 bytes: rank 0 calls it, the launcher broadcasts it */
int  tdde_group_create(tdde_group** out, int32_t n_local, tdde_handle* const* handles, const tdde_shard* shards, const void* nccl_id128);
/* n_steps CN steps on every local shard: c_dev[k] = device state of shard k in ITS local numbering (halo entries are refreshed, owned
 * entries advanced).  g_table as for tdde_propagate.  st (nullable): the job-wide statistics (identical on every rank).  Synchronises. */
int  tdde_group_propagate(tdde_group* g, tdde_c64* const* c_dev, int64_t n_steps, const double* g_table, tdde_stats* st);
void tdde_group_destroy(tdde_group* g);                         /* the handles stay alive and become ordinary handles again */

/* ---- An entry point that allocates nothing (for callers that cannot call cudaMalloc: code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  *out_dev = Re(c^H S c), the total probability of tdde_norm (S: PAPER.md:178-182), computed straight
 * from device copies of the inputs -- no handle, no cudaMalloc / cudaFree / allocating library call.  It is the S-only apply with its
 * fused norm reduction; the per-block partial sums and the completion ticket of that reduction, which the handle path keeps in
 * buffers allocated by tdde_create, live in a file-scope `static __device__` array of TDDE_NOALLOC_MAX_BLOCKS doubles (+ ticket;
 * 64 KB + 256 B that every GPU which loads the library holds until exit).  One block reduces TDDE_NOALLOC_ELEMS_PER_BLOCK elements, so
 *     n_ang * n_rad <= TDDE_NOALLOC_MAX_N = 16 777 216 elements       (BASELINE "large", 6e6, fits; the HBM-scale config does not);
 * larger problems are rejected with TDDE_EINVAL and a text in tdde_last_cuda_error() that names the limit.
 *   S_band_dev : device [n_cls][n_rad][2*w0+1], the row-band layout of tdde_create;  cls_dev : device int32 [n_ang], values in [0, n_cls)
 *   c_dev      : device, n complex128, boundary layout;  out_dev : device double[1];  cuda_stream : cudaStream_t (as void*)
 * w0 <= 32.  Does not synchronise; *out_dev is valid when the stream reaches the end of the call's work.
 * EVERY call on a device shares the one scratch array, which keeps the last call's contents: the call clears the ticket itself (a
 * memset node, no allocation) and overwrites every partial it reads, but two calls that overlap on the GPU (different streams, or two
 * graphs replayed concurrently) race on it -- serialise them.  tdde_snorm_noalloc_setup() resolves the array's device address
 * (cudaGetSymbolAddress, once per device, on the current device); the entry point does the same on its first call on a device, so call
 * the set-up once before capturing a graph.  Errors: TDDE_EINVAL, TDDE_ECUDA. */
#define TDDE_NOALLOC_ELEMS_PER_BLOCK 2048
#define TDDE_NOALLOC_MAX_BLOCKS 8192
#define TDDE_NOALLOC_MAX_N ((int64_t)TDDE_NOALLOC_ELEMS_PER_BLOCK * TDDE_NOALLOC_MAX_BLOCKS)
int tdde_snorm_noalloc_setup(void);
int tdde_snorm_noalloc(int32_t n_ang, int32_t n_rad, int32_t n_cls, int32_t w0, const tdde_c64* S_band_dev, const int32_t* cls_dev,
                       const tdde_c64* c_dev, double* out_dev, void* cuda_stream);

/* Which operator-apply kernel the handle uses: 1 = banded A_L held in registers, 2 = general sparse A_L staged in shared memory
 * (x tile by TMA), 0 = unstaged generic CSR fall-back. */
int tdde_apply_path(const tdde_handle* h);

void        tdde_destroy(tdde_handle* h);          /* NULL is allowed */
const char* tdde_strerror(int status);             /* static string */
const char* tdde_last_cuda_error(void);            /* text of the last CUDA failure seen by this thread */
int         tdde_version(void);                    /* ABI version, currently 2 */

#ifdef __cplusplus
}
#endif
#endif /* TDDE_H_ */
