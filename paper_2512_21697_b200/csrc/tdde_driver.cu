// tdde_driver.cu -- the Crank-Nicolson / BiCGSTAB step driver and the remaining C-ABI entry points.
//
// Control flow without a host sync per iteration (SURVEY 7 hard part 3): every step enqueues its two
// start-of-step applies, `nspec` speculated BiCGSTAB iterations and a one-thread "close" kernel.  Kernels of
// an iteration are no-ops once the device-side `done` flag is set; if the speculated iterations were not
// enough, close latches `stalled`, every later kernel (including later steps) becomes a no-op, and the host
// finds out at its next state read (once per batch of steps), resumes that step with more iterations and
// raises nspec.  All BiCGSTAB scalars stay in SolverState on the device.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "tdde_handle.h"

static const cplx* blk_ptr(const tdde_handle* h, int blk) {
  switch (blk) {
    case BLK_S: return h->d_S;
    case BLK_H0: return h->d_H0;
    case BLK_MP: return h->d_Mp;
    default: return h->d_blk_tmp;
  }
}

int enqueue_apply(tdde_handle* h, const cplx* x, cplx* y, const cplx* aux, int blk, cplx beta, bool with_terms,
                  const double* g_dev, const int* step_ptr, int guard, int fin, SolverState* st, const cplx* addv, int emode, cplx oscale, cplx* y2) {
  ApplyArgs a;
  std::memset(&a, 0, sizeof(a));
  a.x = x; a.y = y; a.aux = aux;
  a.emode = emode; a.oscale = oscale; a.y2 = y2;
  a.addv = (h->path == 1 && h->use_subst && with_terms && h->cfg.n_terms > 0) ? addv : nullptr;
  a.n_ang = h->cfg.n_ang; a.n_rad = h->cfg.n_rad; a.ld = h->ld;
  a.seg_len = (with_terms && h->cfg.n_terms > 0) ? h->seg_len : h->seg_len_s;
  a.cls = h->d_cls;
  a.beta = beta;
  a.g = g_dev; a.step_ptr = step_ptr;
  a.w0 = h->cfg.w0;
  a.guard = guard;
  a.red.partials = h->d_partials; a.red.ticket = h->d_ticket; a.red.st = st; a.red.fin = fin;
  a.red.shard_out = (h->shard_sums && fin != FIN_NONE) ? h->shard_sums : nullptr;
  a.own_lo = h->own_lo; a.own_hi = h->own_hi > 0 ? h->own_hi : h->ld;
  const int T = with_terms ? h->cfg.n_terms : 0;
  a.n_terms = T;
  if (T == 0 && h->have_xmaps) {
    const cplx* vv[9] = {h->X, h->r, h->rhat, h->p, h->v, h->s, h->t, h->y, h->z};
    for (int q = 0; q < 9; ++q)
      if (vv[q] == x) { a.xmap = h->xmaps[q]; a.use_xmap = 1; }
  }
  int rc;
  const bool banded = (h->path == 1);
  if (banded) {
    a.blk = blk_ptr(h, blk);
    a.Rall = h->d_Rall; a.slot = h->d_slot; a.cta_cls = h->d_cta_cls;
    a.Aoff = h->d_Aoff;
    rc = -1;
    if (a.addv && T > 0 && (emode == 0 || emode == 3) && h->seg_len_m > 0) {      // y = addv + coupling terms: DMMA variant
      a.Rfrag = h->d_Rfrag;
      a.seg_len = h->seg_len_m;
      if (h->nbrL || h->nbrR) {                                   // sharded: halo columns straight from the neighbours' copy of this vector
        const cplx* mine[9] = {h->X, h->r, h->rhat, h->p, h->v, h->s, h->t, h->y, h->z};
        int idx = -1;
        for (int q = 0; q < 9; ++q) if (mine[q] == x) idx = q;
        auto pick = [&](tdde_handle* n) -> const cplx* {
          const cplx* theirs[9] = {n->X, n->r, n->rhat, n->p, n->v, n->s, n->t, n->y, n->z};
          return theirs[idx];
        };
        if (idx >= 0 && h->nbrL) { a.xL = pick(h->nbrL); a.ldL = h->nbrL->ld; a.shiftL = h->shiftL; }
        if (idx >= 0 && h->nbrR) { a.xR = pick(h->nbrR); a.ldR = h->nbrR->ld; a.shiftR = h->shiftR; }
      }
      rc = launch_apply_mma(a, T, h->bM0, h->bMS, h->bW, h->stream);
      if (rc == -1) a.seg_len = h->seg_len;
    }
    if (rc == -1) rc = launch_apply_banded(a, T, h->bM0, h->bMS, h->bW, h->apply_ng, h->stream);
  } else if (h->path == 2) {
    a.blk = blk_ptr(h, blk);
    a.Rall = h->d_Rall; a.slot = h->d_slot; a.cta_cls = h->d_cta_cls;
    a.sp_val = h->d_spval; a.sp_col = h->d_spcol;
    a.sp_nslots = 0;
    for (int L = 0; L < T; ++L) { a.sp_nslot[L] = h->sp_nslot[L]; a.sp_nslots += h->sp_nslot[L]; }
    a.sp_xw = h->sp_xw; a.sp_full = h->sp_full; a.sp_reach = h->sp_reach; a.sp_a_smem = h->sp_a_smem;
    rc = launch_apply_sparse(a, h->spW, h->stream);
  } else {
    a.blk_row = blk_ptr(h, blk);
    for (int L = 0; L < T; ++L) {
      a.Rrow[L] = h->d_R[L]; a.w[L] = h->w[L];
      a.A_rowptr[L] = h->d_Arowptr[L]; a.A_col[L] = h->d_Acol[L]; a.A_val[L] = h->d_Aval[L];
    }
    rc = launch_apply_generic(a, h->num_sms, h->stream);
  }
  if (rc == -2) return tdde_cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(apply)");
  if (rc < 0) return TDDE_EINVAL;
  h->launches += rc;
  return 0;
}

static PrecArgs make_prec_args(tdde_handle* h, const cplx* x, cplx* y, const SolverState* st);

// The p-update / s-update of an iteration; when the partitioned solve follows, fused with its spike products (k_vec_spikes).
int enqueue_vec_update(tdde_handle* h, int mode, SolverState* st, bool* fused) {
  static const bool no_fuse = std::getenv("TDDE_NO_VEC_FUSE") != nullptr;
  *fused = false;
  // Below ~2M elements the column-walking fused kernel is latency-bound and loses to the flat update plus the separate spike
  // kernel (measured: Medium 0.390 -> 0.402 ms per step; Large 1.615 -> 1.588, HBM-scale 8.81 -> 8.56)
  if (!no_fuse && h->nint >= (1LL << 21)) {
    const cplx* rhs = mode == 0 ? h->p : h->s;
    int rc = launch_vec_spikes(make_vec_args(h, st, mode == 0 ? FIN_NONE : FIN_S), make_prec_args(h, rhs, nullptr, st), mode, h->stream);
    if (rc == -2) return tdde_cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(vec_spikes)");
    if (rc > 0) { h->launches += rc; *fused = true; return 0; }
  }
  if (mode == 0) h->launches += launch_vec_p(make_vec_args(h, st, FIN_NONE), h->stream);
  else h->launches += launch_vec_s(make_vec_args(h, st, FIN_S), h->stream);
  return 0;
}

int enqueue_precond(tdde_handle* h, const cplx* x, cplx* y, const SolverState* st, bool spikes_done) {
  PrecArgs p = make_prec_args(h, x, y, st);
  p.spikes_done = spikes_done ? 1 : 0;
  int rc = launch_precond(p, h->stream);
  if (rc == -2) return tdde_cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(precond)");
  if (rc < 0) return TDDE_EINVAL;
  h->launches += rc;
  return 0;
}

static PrecArgs make_prec_args(tdde_handle* h, const cplx* x, cplx* y, const SolverState* st) {
  PrecArgs p;
  p.x = x; p.y = y; p.n_ang = h->cfg.n_ang; p.n_rad = h->cfg.n_rad; p.ld = h->ld; p.w = h->cfg.w0;
  p.cls = h->d_cls; p.Lcol = h->d_Lcol; p.Ucol = h->d_Ucol; p.st = st;
  p.slot = h->d_pslot; p.warp_cls = h->d_warp_cls;
  p.P = h->pc_P; p.tile_rows = h->pc_tile_rows; p.int_base = h->pc_base; p.int_rem = h->pc_rem;
  p.Wsp = h->d_Wsp; p.Corner = h->d_Corner; p.Schur = h->d_Schur; p.rsm = h->d_rsm; p.rsp = h->d_rsp;
  p.aslot = h->d_slot; p.cta_cls = h->d_cta_cls;
  p.spikes_done = 0;
  return p;
}

const double* map_g(const tdde_handle* h, const double* g, long long rows, std::vector<double>& buf) {
  if (h->g_identity || !g) return g;
  const int Tu = h->user_terms, Ti = h->cfg.n_terms;
  buf.assign((size_t)rows * Ti, 0.0);
  for (long long r = 0; r < rows; ++r)
    for (int L = 0; L < Tu; ++L) buf[(size_t)r * Ti + h->term_slot[L]] = g[(size_t)r * Tu + L];
  return buf.data();
}

VecArgs make_vec_args(tdde_handle* h, SolverState* st, int fin) {
  VecArgs a;
  a.n = h->nint;
  a.x = h->X; a.r = h->r; a.rhat = h->rhat; a.p = h->p; a.v = h->v; a.s = h->s; a.t = h->t; a.y = h->y; a.z = h->z;
  a.b = h->s;   // start of step: S c lands in the s buffer, H c in the t buffer (both free until the iteration)
  a.u = h->t;
  a.dt = h->cfg.dt;
  a.red.partials = h->d_partials; a.red.ticket = h->d_ticket; a.red.st = st; a.red.fin = fin;
  a.red.shard_out = (h->shard_sums && fin != FIN_NONE) ? h->shard_sums : nullptr;
  return a;
}

int sync_state(tdde_handle* h) {
  CU(cudaMemcpyAsync(h->h_st, h->d_st, sizeof(SolverState), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return 0;
}

// The two start-of-step applies and the initial residual (SURVEY 8(a) a2 + a3): with x0 = c,
//   b = S c - i tau H c,   r0 = b - (S c + i tau H c) = -i dt H c,   hence b = S c + r0 / 2,
// so one H-apply (writing r0 and rhat) and one S-apply (accumulating ||b||^2, storing nothing) give everything.
static int enqueue_step_start(tdde_handle* h) {
  SolverState* st = h->d_st;
  const cplx one = make_double2(1.0, 0.0);
  int rc;
  if (h->split_start) {
    // Shapes with a DMMA apply: one HBM-bound pass gives the block parts  r = -i dt H0 c  and  s = S c,  then the DMMA apply adds the
    // coupling part in place, r = rhat = r + (-i dt) sum_L g_L (A_L (x) R_L) c, and forms ||b||^2 = ||S c + r0 / 2||^2 and ||r0||^2
    ApplyArgs a;
    std::memset(&a, 0, sizeof(a));
    a.x = h->X; a.y = h->r; a.y2 = h->s; a.oscale = make_double2(0.0, -h->cfg.dt);
    a.n_ang = h->cfg.n_ang; a.n_rad = h->cfg.n_rad; a.ld = h->ld; a.seg_len = h->seg_len_s;
    a.cls = h->d_cls; a.blk = h->d_H0; a.slot = h->d_slot; a.cta_cls = h->d_cta_cls; a.n_cta_cls = std::min(h->cta_cls_max, 4);   // at most 4 classes staged per CTA: smaller stages, more CTAs per SM
    if (const char* env = std::getenv("TDDE_B2_NCLS")) a.n_cta_cls = std::max(0, std::min(TDDE_AP_MAXC, std::atoi(env)));
    a.guard = 2; a.red.st = st;
    a.own_lo = h->own_lo; a.own_hi = h->own_hi > 0 ? h->own_hi : h->ld;
    if (h->have_xmaps) { a.xmap = h->xmaps[0]; a.use_xmap = 1; }      // X is work vector 0
    rc = launch_block_dual(a, h->d_S, h->bW, h->stream);
    if (rc == -2) return tdde_cuda_fail(cudaGetLastError(), "cudaFuncSetAttribute(block_dual)");
    if (rc > 0) {
      h->launches += rc;
      return enqueue_apply(h, h->X, h->r, h->s, BLK_H0, make_double2(0.0, -h->cfg.dt), true, h->d_g, &st->step_idx, 2, FIN_R0, st, h->r, 3,
                           one, h->rhat);
    }
  }
  // r0 = rhat = -i dt H c and ||r0||^2, written by the H-apply itself
  if ((rc = enqueue_apply(h, h->X, h->r, nullptr, BLK_H0, one, true, h->d_g, &st->step_idx, 2, FIN_RES0, st, nullptr, 1,
                          make_double2(0.0, -h->cfg.dt), h->rhat)))
    return rc;
  // ||b||^2 = ||S c + r0 / 2||^2 accumulated by the S-apply, which stores nothing; then the start-of-solve scalars
  if ((rc = enqueue_apply(h, h->X, h->s, h->r, BLK_S, one, false, h->d_zero_g, nullptr, 2, FIN_R0S, st, nullptr, 2)))
    return rc;
  return 0;
}

// One full BiCGSTAB iteration in the order of SURVEY 8(c) C4.
// Banded path: since y = M^-1 p, A y = (M + i tau sum_L g_L A_L (x) R_L) y = p + i tau (coupling terms) y up to the rounding
// of the solve, so the two applies of the iteration skip the block part and add p (resp. s) instead.
static int enqueue_iteration(tdde_handle* h) {
  SolverState* st = h->d_st;
  const cplx itau = make_double2(0.0, h->tau);
  int rc;
  bool fused = false;
  if ((rc = enqueue_vec_update(h, 0, st, &fused))) return rc;                             // p = r + beta (p - omega v)
  if ((rc = enqueue_precond(h, h->p, h->y, st, fused))) return rc;                        // y = M^-1 p
  if ((rc = enqueue_apply(h, h->y, h->v, h->rhat, BLK_MP, itau, true, h->d_g, &st->step_idx, 1, FIN_ALPHA, st, h->p))) return rc;
  if ((rc = enqueue_vec_update(h, 1, st, &fused))) return rc;                             // s = r - alpha v, ||s||
  h->launches += launch_vec_halfexit(make_vec_args(h, st, FIN_NONE), h->stream);          // x += alpha y on the ||s|| exit
  if ((rc = enqueue_precond(h, h->s, h->z, st, fused))) return rc;                        // z = M^-1 s
  if ((rc = enqueue_apply(h, h->z, h->t, h->s, BLK_MP, itau, true, h->d_g, &st->step_idx, 1, FIN_OMEGA, st, h->s))) return rc;
  h->launches += launch_vec_xr(make_vec_args(h, st, FIN_R), h->stream);                   // x, r updates, ||r||, <rhat,r>
  return 0;
}

int upload_g(tdde_handle* h, const double* g_table, long long n_steps) {
  const int T = h->cfg.n_terms;
  const long long n_req = n_steps;
  if (T == 0) { if (!h->d_g) { CU(cudaMalloc((void**)&h->d_g, sizeof(double))); h->g_cap = 1; } return 0; }
  if (n_steps > h->g_cap) {
    n_steps = std::max<long long>(n_steps, 4096);       // generous: a new table address would force a re-capture
    if (h->d_g) { CU(cudaStreamSynchronize(h->stream)); cudaFree(h->d_g); h->d_g = nullptr; }
    CU(cudaMalloc((void**)&h->d_g, (size_t)n_steps * T * sizeof(double)));
    h->g_cap = n_steps;
    n_steps = n_req;
  }
  CU(cudaMemcpyAsync(h->d_g, g_table, (size_t)n_steps * T * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  return 0;
}

void fill_stats(const tdde_handle* h, tdde_stats* st) {
  if (!st) return;
  const SolverState* s = h->h_st;
  st->steps = s->steps_done; st->half_iters = s->total_half; st->applies = s->applies; st->preconds = s->preconds;
  st->rel_res = s->last_rel_res; st->status = s->status; st->last_half_iters = s->last_half_iters;
}

static int enqueue_step_raw(tdde_handle* h) {
  int rc;
  if ((rc = enqueue_step_start(h))) return rc;
  for (int it = 0; it < h->nspec; ++it)
    if ((rc = enqueue_iteration(h))) return rc;
  h->launches += launch_step_close(h->d_st, h->stream);
  return 0;
}

// One step as a CUDA graph.  The sequence is identical for every step (the g row is picked by the device-side step
// counter), so it is captured once and replayed; any failure falls back to plain launches for good.
static bool ensure_graph(tdde_handle* h) {
  static const bool disabled = std::getenv("TDDE_NO_GRAPH") != nullptr;
  if (disabled || !h->graph_ok || !h->nspec_learned) return false;
  if (!h->step_exec || h->graph_nspec != h->nspec || h->graph_g != h->d_g) {
    if (h->step_exec) { cudaGraphExecDestroy(h->step_exec); h->step_exec = nullptr; }
    if (!h->cap && cudaStreamCreateWithFlags(&h->cap, cudaStreamNonBlocking) != cudaSuccess) { h->graph_ok = false; cudaGetLastError(); return false; }
    cudaStream_t user = h->stream;
    const long long l0 = h->launches;
    cudaGraph_t g = nullptr;
    bool ok = cudaStreamBeginCapture(h->cap, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
      h->stream = h->cap;
      ok = enqueue_step_raw(h) == 0;
      h->stream = user;
      ok = (cudaStreamEndCapture(h->cap, &g) == cudaSuccess) && ok && g;
    }
    h->graph_launches = h->launches - l0;
    h->launches = l0;
    if (ok) ok = cudaGraphInstantiate(&h->step_exec, g, 0) == cudaSuccess;
    if (g) cudaGraphDestroy(g);
    if (!ok) { h->graph_ok = false; h->step_exec = nullptr; cudaGetLastError(); return false; }
    h->graph_nspec = h->nspec; h->graph_g = h->d_g;
  }
  return true;
}

static int enqueue_step(tdde_handle* h) {
  if (!ensure_graph(h)) return enqueue_step_raw(h);
  CU(cudaGraphLaunch(h->step_exec, h->stream));
  h->launches += h->graph_launches;
  return 0;
}

// X (internal layout) holds c; advance n_steps steps.  Always ends with one state read.
static int run_steps(tdde_handle* h, long long n_steps) {
  long long enq = 0;          // steps enqueued so far (== steps_done when nothing stalled)
  int rc;
  h->launches += launch_step_open(h->d_st, 0, 0, 0, h->stream);
  while (true) {
    const long long batch = h->nspec_learned ? 64 : 4;      // short batches until nspec has settled
    const long long upto = std::min(n_steps, enq + batch);
    for (; enq < upto; ++enq) {
      if ((rc = enqueue_step(h))) return rc;
    }
    if ((rc = sync_state(h))) return rc;
    CU(cudaGetLastError());
    if (h->h_st->status != 0) return h->h_st->status;
    while (h->h_st->stalled) {
      // the step after steps_done ran out of speculated iterations: resume it
      h->launches += launch_step_open(h->d_st, 0, 0, 1, h->stream);
      const int more = std::max(2, h->nspec);
      for (int it = 0; it < more; ++it)
        if ((rc = enqueue_iteration(h))) return rc;
      h->launches += launch_step_close(h->d_st, h->stream);
      if ((rc = sync_state(h))) return rc;
      if (h->h_st->status != 0) return h->h_st->status;
      if (!h->h_st->stalled) {
        const int need = (h->h_st->last_half_iters + 1) / 2;
        h->nspec = std::min(h->cfg.max_iter, std::max(h->nspec, need));
      }
      enq = h->h_st->steps_done;      // steps after the stalled one were no-ops: redo them
    }
    if (!h->h_st->stalled && h->h_st->steps_done >= upto) h->nspec_learned = true;
    if (h->h_st->steps_done >= n_steps) { ensure_graph(h); return 0; }   // capture now, outside the next call's steps
    enq = h->h_st->steps_done;
  }
}

extern "C" int tdde_propagate(tdde_handle* h, tdde_c64* c_dev, int64_t n_steps, const double* g_table, tdde_stats* st) {
  if (!h || !c_dev || n_steps < 0 || (n_steps > 0 && h->user_terms > 0 && !g_table)) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  std::vector<double> gbuf;
  g_table = map_g(h, g_table, n_steps, gbuf);
  if (st) std::memset(st, 0, sizeof(*st));
  if (n_steps == 0) return 0;
  int rc;
  if ((rc = upload_g(h, g_table, n_steps))) return rc;
  // a failure latched by an earlier call is cleared here: each call reports its own status
  h->h_st->status = 0; h->h_st->stalled = 0; h->h_st->done = 1; h->h_st->force = 0;
  h->h_st->rtol2 = h->cfg.rtol * h->cfg.rtol; h->h_st->max_half = 2 * h->cfg.max_iter;
  CU(cudaMemcpyAsync(h->d_st, h->h_st, sizeof(SolverState), cudaMemcpyHostToDevice, h->stream));
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(c_dev), h->X, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  rc = run_steps(h, n_steps);
  h->launches += launch_to_boundary(h->X, reinterpret_cast<cplx*>(c_dev), h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  CU(cudaStreamSynchronize(h->stream));
  fill_stats(h, st);
  return rc;
}

extern "C" int tdde_step(tdde_handle* h, tdde_c64* c_dev, const double* g_mid, tdde_stats* st) {
  return tdde_propagate(h, c_dev, 1, g_mid, st);
}

extern "C" int tdde_propagate_host(tdde_handle* h, tdde_c64* c_host, int64_t n_steps, const double* g_table, tdde_stats* st) {
  if (!h || !c_host) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  const size_t bytes = (size_t)h->n * sizeof(cplx);
  if (!h->c_stage) CU(cudaMalloc((void**)&h->c_stage, bytes));
  CU(cudaMemcpyAsync(h->c_stage, c_host, bytes, cudaMemcpyHostToDevice, h->stream));
  int rc = tdde_propagate(h, reinterpret_cast<tdde_c64*>(h->c_stage), n_steps, g_table, st);
  CU(cudaMemcpyAsync(c_host, h->c_stage, bytes, cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return rc;
}

#ifdef TDDE_WITH_BENCH
extern "C" int tdde_step_forced(tdde_handle* h, tdde_c64* c_dev, const double* g_mid, int32_t n_iters, tdde_c64* trace_dev) {
  if (!h || !c_dev || n_iters < 0 || (h->user_terms > 0 && !g_mid)) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  std::vector<double> gbuf;
  g_mid = map_g(h, g_mid, 1, gbuf);
  int rc;
  if ((rc = upload_g(h, g_mid, 1))) return rc;
  h->h_st->status = 0; h->h_st->stalled = 0; h->h_st->done = 1;
  CU(cudaMemcpyAsync(h->d_st, h->h_st, sizeof(SolverState), cudaMemcpyHostToDevice, h->stream));
  const int na = h->cfg.n_ang, nr = h->cfg.n_rad;
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(c_dev), h->X, na, nr, h->ld, h->stream);
  h->launches += launch_step_open(h->d_st, 0, 1, 0, h->stream);
  if ((rc = enqueue_step_start(h))) return rc;
  for (int it = 0; it < n_iters; ++it) {
    if ((rc = enqueue_iteration(h))) return rc;
    if (trace_dev) {
      const cplx* vecs[8] = {h->p, h->v, h->s, h->t, h->X, h->r, h->y, h->z};
      for (int q = 0; q < 8; ++q) {
        cplx* dst = reinterpret_cast<cplx*>(trace_dev) + ((size_t)it * 8 + q) * (size_t)h->n;
        h->launches += launch_to_boundary(vecs[q], dst, na, nr, h->ld, h->stream);
      }
    }
  }
  h->launches += launch_to_boundary(h->X, reinterpret_cast<cplx*>(c_dev), na, nr, h->ld, h->stream);
  if ((rc = sync_state(h))) return rc;
  const int status = h->h_st->status;
  // leave the state idle and unforced for the next call
  h->h_st->status = 0; h->h_st->force = 0; h->h_st->done = 1;
  CU(cudaMemcpyAsync(h->d_st, h->h_st, sizeof(SolverState), cudaMemcpyHostToDevice, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  return status;
}

#endif  // TDDE_WITH_BENCH

extern "C" int tdde_norm(tdde_handle* h, const tdde_c64* c_dev, double* out) {
  if (!h || !c_dev || !out) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  int rc;
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(c_dev), h->y, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  if ((rc = enqueue_apply(h, h->y, h->z, h->y, BLK_S, make_double2(0, 0), false, h->d_zero_g, nullptr, 0, FIN_NORM, h->d_st))) return rc;
  if ((rc = sync_state(h))) return rc;
  *out = h->h_st->norm_out;
  return 0;
}

extern "C" int tdde_apply(tdde_handle* h, tdde_c64 alpha, tdde_c64 beta, const double* g, const tdde_c64* x_dev, tdde_c64* y_dev) {
  if (!h || !x_dev || !y_dev || x_dev == y_dev || (h->user_terms > 0 && !g)) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  std::vector<double> gbuf;
  g = map_g(h, g, 1, gbuf);
  int rc;
  if (h->cfg.n_terms > 0)
    CU(cudaMemcpyAsync(h->d_g_small, g, h->cfg.n_terms * sizeof(double), cudaMemcpyHostToDevice, h->stream));
  h->launches += launch_combine_blocks(h->d_S, h->d_H0, make_double2(alpha.re, alpha.im),
                                       make_double2(beta.re, beta.im), h->d_blk_tmp, h->blk_count, h->stream);
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(x_dev), h->y, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  if ((rc = enqueue_apply(h, h->y, h->z, nullptr, BLK_TMP, make_double2(beta.re, beta.im), true, h->d_g_small, nullptr, 0, FIN_NONE, h->d_st))) return rc;
  h->launches += launch_to_boundary(h->z, reinterpret_cast<cplx*>(y_dev), h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  CU(cudaGetLastError());
  return 0;
}

extern "C" int tdde_precond(tdde_handle* h, const tdde_c64* x_dev, tdde_c64* y_dev) {
  if (!h || !x_dev || !y_dev) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  int rc;
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(x_dev), h->y, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  if ((rc = enqueue_precond(h, h->y, h->z, nullptr))) return rc;
  h->launches += launch_to_boundary(h->z, reinterpret_cast<cplx*>(y_dev), h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  CU(cudaGetLastError());
  return 0;
}
