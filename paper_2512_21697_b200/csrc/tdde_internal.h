// tdde_internal.h -- private declarations shared by the host API and the kernel translation units.
//
// Internal layout ("channel-fastest"): element (radial j, channel a) of a vector lives at X[j * ld + a],
// ld = n_ang rounded up to a multiple of 32.  Lanes of a warp then own consecutive channels: radial band
// coefficients R_L[i][j] are warp-uniform, the angular coefficients A_L[a'][a'+o] are per-lane registers
// and the vector accesses are coalesced 16-byte loads.  Pad channels (a >= n_ang) hold zeros throughout.
// The boundary layout (tdde.h) is channel-major; transposes happen at entry/exit of the API calls.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include "tdde.h"
#ifdef TDDE_WITH_BENCH
#include "tdde_bench.h"
#endif

#define TDDE_MAX_TERMS 24
#define TDDE_MAX_PARTIAL_BLOCKS 65536
#define TDDE_TINY 1e-290
#ifndef TDDE_AP_NC
#define TDDE_AP_NC 128     // banded apply: channels per CTA
#endif
#ifndef TDDE_AP_MINB
#define TDDE_AP_MINB 2     // banded apply: CTAs per SM the kernel is compiled for
#endif
#ifndef TDDE_AP_MINB2
#define TDDE_AP_MINB2 1    // CTAs per SM for the two-group (256-thread) variant
#endif
#ifndef TDDE_AP_JC
#define TDDE_AP_JC 4       // banded apply: radial rows per pipeline stage
#endif
#ifndef TDDE_AP_RU
#define TDDE_AP_RU 2
#endif
#ifndef TDDE_AP_RU9
#define TDDE_AP_RU9 1    // rows unrolled together for W >= 9
#endif
#ifndef TDDE_AP_MAXC
#define TDDE_AP_MAXC 16    // banded apply: distinct kappa-classes per CTA staged in shared memory
#endif
#define TDDE_PC_MAXC 2      // preconditioner: distinct kappa-classes per warp staged in shared memory
// half-bandwidths the preconditioner kernels are instantiated for (others <= 32 take the runtime-w two-sweep kernel)
#define TDDE_PC_WIDTHS(X) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12) X(13)
#define TDDE_PC_MAXW 13

typedef double2 cplx;

// ---- device-resident solver state: every BiCGSTAB scalar and flag lives here ----
struct SolverState {
  cplx rho, rho_old, alpha, omega, beta;   // C4 notation
  double nb2;          // ||b||^2
  double res2;         // ||r||^2 or ||s||^2 of the latest test
  double rtol2;        // rtol^2
  double norm_out;     // tdde_norm result
  int done;            // this step's solve finished (converged or failed)
  int status;          // latched tdde_status (0 = ok)
  int stalled;         // speculated iterations ran out before convergence; later kernels are no-ops
  int half_exit;       // 1: ||s|| exit taken and x += alpha y still pending; 2: applied
  int first;           // first iteration of the step: p = r
  int force;           // exit tests disabled (tdde_step_forced)
  int half_iters;      // of the current step
  int max_half;        // 2 * max_iter
  int step_idx;        // index into the device g table of the step being solved
  int pad0;
  long long steps_done, total_half, applies, preconds;
  int last_half_iters;
  int pad1;
  double last_rel_res;
};

// finalisation codes: what the last block does with the reduced sums (d0 complex, d1 real)
enum FinCode {
  FIN_NONE = 0,
  FIN_NB,      // nb2 = d1
  FIN_ALPHA,   // d0 = <rhat, v>  -> alpha = rho / d0
  FIN_OMEGA,   // d0 = <s, t>, d1 = <t,t>  -> omega = conj(d0) / d1
  FIN_NORM,    // norm_out = Re d0
  FIN_R0,      // d0.x = ||b||^2, d1 = ||r0||^2 -> rho, init, zero-iteration exit
  FIN_S,       // d1 = ||s||^2 -> half-step exit test
  FIN_R,       // d0 = <rhat, r>, d1 = ||r||^2 -> convergence test, rho, beta
  FIN_RES0,    // d1 = ||r0||^2 (start of step, from the H-apply that writes r0 and rhat): res2 = d1
  FIN_R0S,     // d1 = ||b||^2 (start of step, from the S-apply): the FIN_R0 logic with ||r0||^2 taken from res2
  FIN_DOTS     // test export: rho_old = d0, res2 = d1, nothing else
};

struct ReduceCtx {
  double* partials;        // [TDDE_MAX_PARTIAL_BLOCKS][4]
  unsigned int* ticket;    // zero between kernels
  SolverState* st;
  int fin;
  double* shard_out;       // channel-slab sharding (tdde_shard.cu): the last block writes its three sums here and does NOT finalise;
                           //   the sums are all-reduced over the ranks and k_finalize applies them.  nullptr = single GPU
};

// ---- operator apply ----
struct ApplyArgs {
  CUtensorMap xmap;        // 2-D tensor map of x ([n_rad][2 ld] doubles, box 256 x TDDE_AP_JC), valid iff use_xmap
  int use_xmap;            // T == 0 kernel only: fetch the x tile of a stage with one tensor TMA copy
  const cplx* x;           // internal layout
  cplx* y;
  const cplx* aux;         // vector for the fused dot (nullable)
  int emode;               // write-out: 0 y = result; 1 y = y2 = oscale * result (r0 and rhat); 3 (k_apply_mma) y = y2 = result,
                           //   d0.x accumulates |aux + result / 2|^2 (||b||^2 with aux = S c), d1 = ||result||^2; 2 nothing stored,
                           //   d1 accumulates |result + aux / 2|^2 (||b||^2 with aux = r0, R6)
  cplx oscale;
  cplx* y2;
  const cplx* addv;        // banded path, nullable: y = addv + (coupling terms only) x; the block part is skipped
  int n_ang, n_rad, ld;
  int seg_len;             // radial rows per thread
  const int* cls;          // [ld] class per channel (pads: class 0)
  const cplx* blk;         // column-band block coefficients [n_cls][n_rad][2w0+1]: blk[k][j][e] = M_k[j-w0+e][j]
  cplx beta;               // multiplies every coupling term
  const double* g;         // device g table
  const int* step_ptr;     // nullable: row of g = *step_ptr
  int n_terms;
  const cplx* Rall;        // banded path: column-band of every term interleaved [n_rad][T][2w+1]: Rall[j][L][e] = R_L[j-w+e][j]
  const int* slot;         // [ld] index of the channel's class in its CTA's class list, -1 = not staged
  const int* cta_cls;      // [n_cta][TDDE_AP_MAXC] classes staged per CTA (-1 = unused)
  int n_cta_cls;           // k_block_dual: the largest number of classes any CTA stages (sizes its shared-memory stage)
  const cplx* Aoff;        // banded path: [n_slots][ld], slot = (term, offset) in kernel order
  const double* Rfrag;     // DMMA path (tdde_apply_mma.cu): B-operand fragments of every 4-row slice, nullable
  // staged sparse-A path (tdde_apply_sparse.cu): ELL rows of every term, slot-major [sp_nslots][ld]; blk and Rall padded to 2W+1
  const cplx* sp_val;
  const int* sp_col;       // absolute internal channel index (own channel for padding slots)
  int sp_nslot[TDDE_MAX_TERMS];
  int sp_nslots;           // sum of sp_nslot
  int sp_xw;               // channels of the staged x tile
  int sp_full;             // 1: the tile is the whole row (sp_xw == ld)
  int sp_reach;            // otherwise: largest |column - row| over all terms; tile = 128 + 2 reach channels
  int sp_a_smem;           // 1: the ELL rows of the CTA's channels are copied to shared memory once; 0: read from global (L1/L2) per row
  // generic path
  const int* A_rowptr[TDDE_MAX_TERMS];
  const int* A_col[TDDE_MAX_TERMS];
  const cplx* A_val[TDDE_MAX_TERMS];
  const cplx* Rrow[TDDE_MAX_TERMS];   // row-band [n_rad][2w+1] as at the boundary
  const cplx* blk_row;     // row-band block coefficients [n_cls][n_rad][2w0+1]
  int w[TDDE_MAX_TERMS];
  int w0;
  // k_apply_mma<GATHER> (sharding): channel a < own_lo of row j is xL[j * ldL + a + shiftL], a >= own_hi is xR[j * ldR + a + shiftR]
  const cplx *xL, *xR;
  int ldL, ldR, shiftL, shiftR;
  int own_lo, own_hi;      // channels [own_lo, own_hi) are written and enter the fused sums (sharding: the owned slab; else 0, ld)
  int guard;               // 0 none; 1: no-op when st->done|stalled|status (iterations); 2: no-op when stalled|status (start of step)
  ReduceCtx red;
};

struct VecArgs {
  long long n;             // internal element count n_rad * ld
  cplx *x, *r, *rhat, *p, *v, *s, *t, *y, *z, *b, *u;
  double dt;               // r0 = -i dt (H c)
  ReduceCtx red;
};

struct PrecArgs {
  const cplx* x;
  cplx* y;
  int n_ang, n_rad, ld, w;
  const int* cls;
  const cplx* Lcol;        // [n_cls][n_rad][w]:  Lcol[k][i][d-1] = L_k[i+d][i]
  const cplx* Ucol;        // [n_cls][n_rad][w+1]: [0] = 1/U_k[i][i], [1] = U_k[i-1][i]/U_k[i][i], [d>=2] = U_k[i-d][i]
  const int* slot;         // [ld] index of the channel's class in its warp's class list, -1 = not staged
  const int* warp_cls;     // [ld/32][TDDE_PC_MAXC] classes staged per warp (-1 = unused)
  // partitioned solve (tdde_partition.h); P == 1: plain LU over all rows
  int P;                   // interiors
  int tile_rows;           // longest interior = rows of the shared-memory tile
  int int_base, int_rem;   // interior q has int_base + (q < int_rem) rows and starts at row q (int_base + w) + min(q, int_rem);
                           // separator q = the w rows after interior q (make_partition_plan)
  const cplx* Wsp;         // [n_cls][n_rad][2w] left spikes
  const cplx* Corner;      // [n_cls][P][2][w][w] corner blocks of A_IS
  const cplx* Schur;       // [n_cls][P-1][3][w][w] block Thomas factors of the Schur complement
  cplx* rsm;               // scratch [P][w][ld]: P1 -> P2: spike products towards the separator before each interior;
                           //   P2 -> P3: A_IS x_S for the first w rows of each interior
  cplx* rsp;               // scratch [P][w][ld]: P1 -> P2: spike products towards the separator after each interior; inside P2 the
                           //   forward-eliminated Schur rhs; P2 -> P3: A_IS x_S for the last w rows of each interior
  const int* aslot;        // [ld] the apply's per-CTA class slot (128-channel groups), used by k_precond_spikes
  const int* cta_cls;      // [n_cta][TDDE_AP_MAXC]
  const SolverState* st;   // nullable guard
  int spikes_done;         // 1: rsm / rsp already hold the spike products of x (formed by k_vec_spikes): skip P1
};

__host__ __device__ inline int pc_lo(const PrecArgs& p, int q) { return q * (p.int_base + p.w) + (q < p.int_rem ? q : p.int_rem); }
__host__ __device__ inline int pc_len(const PrecArgs& p, int q) { return p.int_base + (q < p.int_rem ? 1 : 0); }

int tdde_num_sms();   // multiprocessor count of the current device
// launchers (each returns the number of kernels launched, or -1 if no instantiation fits)
int launch_apply_banded(const ApplyArgs& a, int T, int m0, int mstep, int W, int ng, cudaStream_t s);
bool apply_banded_available(int T, int m0, int mstep, int W);
int apply_banded_shapes(int (*out)[4], int cap);
int launch_apply_generic(const ApplyArgs& a, int num_sms, cudaStream_t s);
// DMMA variant of the in-iteration banded apply (y = addv + coupling terms): shapes, fragment table, launcher
bool apply_mma_available(int T, int m0, int mstep, int W);
int apply_mma_halo(int W);
int apply_mma_channels(int W);
int launch_apply_mma(const ApplyArgs& a, int T, int m0, int mstep, int W, cudaStream_t s);
int launch_block_dual(const ApplyArgs& a, const cplx* blk2, int W, cudaStream_t s);   // y = oscale (blk) x, y2 = (blk2) x
int launch_apply_sparse(const ApplyArgs& a, int W, cudaStream_t s);
size_t apply_sparse_smem(int W, int T, int nslots, int xw, bool a_in_smem);
int launch_precond(const PrecArgs& a, cudaStream_t s);
size_t precond_tile_smem(int w, int tile_rows);
int launch_vec_spikes(const VecArgs& v, const PrecArgs& a, int mode, cudaStream_t s);   // dynamic shared memory of k_precond_tile
int launch_vec_p(const VecArgs& a, cudaStream_t s);
int launch_vec_s(const VecArgs& a, cudaStream_t s);
int launch_vec_halfexit(const VecArgs& a, cudaStream_t s);
int launch_vec_xr(const VecArgs& a, cudaStream_t s);
int launch_step_open(SolverState* st, int step_idx, int force, int clear_stall_only, cudaStream_t s);
int launch_step_close(SolverState* st, cudaStream_t s);
int launch_to_internal(const cplx* c, cplx* X, int n_ang, int n_rad, int ld, cudaStream_t s);
int launch_to_boundary(const cplx* X, cplx* c, int n_ang, int n_rad, int ld, cudaStream_t s);
int launch_combine_blocks(const cplx* S, const cplx* H0, cplx alpha, cplx beta, cplx* out, long long count, cudaStream_t s);
int launch_fill(cplx* v, long long n, unsigned seed, cudaStream_t s);
int launch_dfma_peak(double* out, int blocks, int threads, int iters, cudaStream_t s);
int launch_fp64_pipe_probe(double* out, int blocks, int threads, int iters, int mode, cudaStream_t s);
