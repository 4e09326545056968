// tdde_handle.h -- the opaque handle behind tdde.h and the host-side helpers shared by the API files.
#pragma once
#include <complex>
#include <string>
#include <vector>
#include "tdde_internal.h"

typedef std::complex<double> zc;

struct tdde_handle {
  tdde_config cfg;
  cudaStream_t stream = nullptr;
  int device = 0;                // the device that was current at tdde_create; every entry point runs on it
  int num_sms = 148;             // cudaDevAttrMultiProcessorCount of that device
  int ld = 0;                    // padded channel count (multiple of 32)
  long long nint = 0;            // n_rad * ld
  long long n = 0;               // n_ang * n_rad
  double tau = 0;                // dt / 2

  // apply path
  int path = 0;                  // 1 banded register-A fast path, 2 staged sparse-A path, 0 generic
  int spW = 0, sp_nslots = 0, sp_xw = 0, sp_full = 0, sp_reach = 0, sp_a_smem = 1;   // staged sparse-A path
  int sp_nslot[TDDE_MAX_TERMS] = {};
  cplx* d_spval = nullptr;
  int* d_spcol = nullptr;
  bool use_subst = true;         // banded path: in-iteration applies use A y = p + i tau (coupling) y (needs a benign LU)
  int bT = 0, bM0 = 0, bMS = 0, bW = 0;
  // The banded kernels are instantiated for a few (T, m_L, W) shapes; a problem whose structure FITS inside one (fewer terms, smaller
  // offsets, narrower bands) runs on it with zero-filled slots: internally the handle then has cfg.n_terms = the shape's T, the
  // caller's term L sits in slot term_slot[L], and every g the caller passes is expanded (map_g)
  int user_terms = 0;
  int term_slot[TDDE_MAX_TERMS] = {};
  bool g_identity = true;
  int seg_len = 0;               // radial rows per thread (banded path)
  int seg_len_m = 0;             // radial rows per CTA of the DMMA apply (multiple of 8); 0 = that kernel is not used
  double* d_Rfrag = nullptr;     // its B-operand fragment table
  bool split_start = false;      // start of step = block pass (k_block_dual) + DMMA coupling apply instead of H-apply + S-apply
  int seg_len_s = 0;             // radial rows per thread for the S-only (T = 0) apply: latency-bound, wants more CTAs
  int apply_ng = 1;              // warp groups the terms are split over (banded path)
  bool norm_banded = false;      // S-only apply can use the banded T=0 kernel

  // device constants
  int* d_cls = nullptr;                      // [ld]
  cplx *d_S = nullptr, *d_H0 = nullptr, *d_Mp = nullptr, *d_blk_tmp = nullptr;   // block bands in the path's layout
  long long blk_count = 0;                   // n_cls * n_rad * (2 w0 + 1)
  cplx* d_R[TDDE_MAX_TERMS] = {};            // per term band in the path's layout (col-band or row-band)
  int w[TDDE_MAX_TERMS] = {};
  cplx* d_Aoff = nullptr;                    // banded path
  cplx* d_Rall = nullptr;                    // banded path: [n_rad][T][2w+1]
  int *d_slot = nullptr, *d_cta_cls = nullptr;
  int cta_cls_max = TDDE_AP_MAXC;            // largest number of classes staged by one 128-channel CTA
  int* d_Arowptr[TDDE_MAX_TERMS] = {};       // generic path
  int* d_Acol[TDDE_MAX_TERMS] = {};
  cplx* d_Aval[TDDE_MAX_TERMS] = {};
  cplx *d_Lcol = nullptr, *d_Ucol = nullptr; // preconditioner factors
  int *d_pslot = nullptr, *d_warp_cls = nullptr;
  int pc_P = 1, pc_tile_rows = 0;            // partitioned solve (tdde_partition.h)
  int pc_base = 0, pc_rem = 0;               // interior q: pc_base + (q < pc_rem) rows
  cplx *d_Wsp = nullptr, *d_Corner = nullptr, *d_Schur = nullptr, *d_rsm = nullptr, *d_rsp = nullptr;
  double lu_growth = 1.0;                    // largest element growth of the unpivoted interior LUs over all classes

  // work vectors (internal layout)
  cplx *X = nullptr, *r = nullptr, *rhat = nullptr, *p = nullptr, *v = nullptr, *s = nullptr, *t = nullptr,
       *y = nullptr, *z = nullptr;
  CUtensorMap xmaps[9];                      // per work vector (X, r, rhat, p, v, s, t, y, z), for the S-only apply
  bool have_xmaps = false;
  cplx* c_stage = nullptr;                   // boundary-layout device buffer for tdde_propagate_host

  // observables (tdde_project): eigenvectors [n_cls][n_rad][n_states] and the probability buffer [n_ang][n_states]
  cplx* d_eig = nullptr;
  double* d_proj = nullptr;
  int n_states = 0;

  // channel-slab sharding (tdde_shard.cu): a handle that is one shard of a group owns the local channels
  // [own_lo, own_hi) (the rest are halo inputs) and hands its reduction sums to the group instead of finalising them
  int own_lo = 0, own_hi = 0;                // own_hi == 0: not sharded (all of [0, ld))
  double* shard_sums = nullptr;              // device [4]
  // fused halo gather (k_apply_mma<GATHER>): the shards that own this shard's left / right halo columns and the channel shift into
  // their local numbering; set by tdde_group_create when every shard of the process qualifies
  tdde_handle *nbrL = nullptr, *nbrR = nullptr;
  int shiftL = 0, shiftR = 0;

  // solver state, scratch
  SolverState* d_st = nullptr;
  SolverState* d_st_bench = nullptr;         // never-idle dummy state for tdde_time_kernel
  SolverState* h_st = nullptr;               // pinned mirror
  double* d_partials = nullptr;
  unsigned int* d_ticket = nullptr;
  double* d_g = nullptr;                     // [g_cap][T]
  long long g_cap = 0;
  double* d_g_small = nullptr;               // [T] for tdde_apply
  double* d_zero_g = nullptr;                // [T] zeros
  int nspec = 1;                             // speculated iterations per step (grows when a step stalls)
  bool nspec_learned = false;                // first batches are short until one has passed without a stall
  long long launches = 0;
  // CUDA graph of one step (start + nspec iterations + close): captured once on an internal stream, replayed on the
  // caller's stream; re-captured when nspec or the device g table changes
  cudaStream_t cap = nullptr;
  cudaGraphExec_t step_exec = nullptr;
  int graph_nspec = -1;
  const double* graph_g = nullptr;
  long long graph_launches = 0;
  bool graph_ok = true;
};

// Every entry point runs on the device the handle was created on, whatever the caller's current device is.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// a CUDA event that is destroyed on every exit path
struct ScopedEvent {
  cudaEvent_t e = nullptr;
  cudaError_t create() { return cudaEventCreate(&e); }
  ~ScopedEvent() { if (e) cudaEventDestroy(e); }
  operator cudaEvent_t() const { return e; }
};

extern thread_local std::string g_last_cuda_error;
int tdde_cuda_fail(cudaError_t e, const char* what);

#define CU(call)                                               \
  do {                                                         \
    cudaError_t e__ = (call);                                  \
    if (e__ != cudaSuccess) return tdde_cuda_fail(e__, #call); \
  } while (0)

// enqueue helpers (tdde_driver.cu)
enum BlkSel { BLK_S = 0, BLK_H0 = 1, BLK_MP = 2, BLK_TMP = 3 };
int enqueue_apply(tdde_handle* h, const cplx* x, cplx* y, const cplx* aux, int blk, cplx beta, bool with_terms,
                  const double* g_dev, const int* step_ptr, int guard, int fin, SolverState* st,
                  const cplx* addv = nullptr, int emode = 0, cplx oscale = cplx{1.0, 0.0}, cplx* y2 = nullptr);
int enqueue_precond(tdde_handle* h, const cplx* x, cplx* y, const SolverState* st, bool spikes_done = false);
int enqueue_vec_update(tdde_handle* h, int mode, SolverState* st, bool* fused);   // mode 0: p-update, 1: s-update (+ spike products when fused)
VecArgs make_vec_args(tdde_handle* h, SolverState* st, int fin);
int sync_state(tdde_handle* h);
int upload_g(tdde_handle* h, const double* g_table, long long n_steps);   // g table -> device (grows d_g)
void fill_stats(const tdde_handle* h, tdde_stats* st);                      // from the pinned mirror of the solver state
// g as the caller gives it ([rows][user_terms]) -> as the kernels index it ([rows][cfg.n_terms]); returns g itself when they coincide
bool build_mma_frags(int T, int W, int n_rad, const void* Rall, std::vector<double>& out);   // tdde_apply_mma.cu
const double* map_g(const tdde_handle* h, const double* g, long long rows, std::vector<double>& buf);
