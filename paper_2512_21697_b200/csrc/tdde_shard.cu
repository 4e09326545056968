// tdde_shard.cu -- channel-slab sharding of the CN / BiCGSTAB step over several GPUs.
//
// A shard is an ordinary handle built from the rank-local problem ([halo | owned | halo] channels).  The group enqueues every phase of
// the step on all local shards, then the collective that phase needs:
//   * halo exchange before each apply: the halo columns of the apply's input vector are overwritten with their owners' values
//     (local shards: one strided device copy per piece; remote: pack -> ncclSend / ncclRecv in one group -> unpack);
//   * fused reductions: every reducing kernel runs with ReduceCtx::shard_out set, so its last block leaves the three sums in a
//     device buffer instead of updating the scalars; the buffers are summed over all shards (a tiny kernel locally, ncclAllReduce
//     between ranks) and k_finalize applies finalize_scalars on every shard -- all stream-ordered, no host round trip.
// Sums run over OWNED channels only: the apply kernels write and reduce lanes in [own_lo, own_hi) only, and the halo columns of
// r, rhat, p, v, s, t therefore stay exactly zero (they are zero at attach and every update of them is linear in them), so the
// vector kernels need no mask.  The host reads the solver state once per CN step (the single-GPU driver: once per 64 steps).
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <dlfcn.h>
#include "tdde_handle.h"
#include "tdde_reduce.cuh"

enum ShardVec { SV_X = 0, SV_Y = 1, SV_Z = 2 };

struct HaloPiece { int peer, lo, src_lo, n; };   // recv: [lo, lo+n) here = [src_lo, ..) on peer; send: [lo, lo+n) here goes to peer

// ---- NCCL through dlopen (torch ships libnccl.so.2; no link-time dependency, the single-GPU library never needs it) ----
struct NcclId { char bytes[128]; };
struct NcclApi {
  void* lib = nullptr;
  int (*GetUniqueId)(void*) = nullptr;
  int (*CommInitRank)(void**, int, NcclId, int) = nullptr;
  int (*AllReduce)(const void*, void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*Send)(const void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*Recv)(void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*GroupStart)() = nullptr;
  int (*GroupEnd)() = nullptr;
  int (*CommDestroy)(void*) = nullptr;
};
static const int kNcclFloat64 = 8, kNcclSum = 0;

static NcclApi* nccl_api() {
  static NcclApi api;
  static bool tried = false;
  if (tried) return api.lib ? &api : nullptr;
  tried = true;
  void* lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_NOLOAD);
  if (!lib) lib = dlopen("libnccl.so.2", RTLD_NOW);
  if (!lib) lib = dlopen("libnccl.so", RTLD_NOW);
  if (!lib) return nullptr;
  auto sym = [&](const char* n) { return dlsym(lib, n); };
  api.GetUniqueId = reinterpret_cast<int (*)(void*)>(sym("ncclGetUniqueId"));
  api.CommInitRank = reinterpret_cast<int (*)(void**, int, NcclId, int)>(sym("ncclCommInitRank"));
  api.AllReduce = reinterpret_cast<int (*)(const void*, void*, size_t, int, int, void*, cudaStream_t)>(sym("ncclAllReduce"));
  api.Send = reinterpret_cast<int (*)(const void*, size_t, int, int, void*, cudaStream_t)>(sym("ncclSend"));
  api.Recv = reinterpret_cast<int (*)(void*, size_t, int, int, void*, cudaStream_t)>(sym("ncclRecv"));
  api.GroupStart = reinterpret_cast<int (*)()>(sym("ncclGroupStart"));
  api.GroupEnd = reinterpret_cast<int (*)()>(sym("ncclGroupEnd"));
  api.CommDestroy = reinterpret_cast<int (*)(void*)>(sym("ncclCommDestroy"));
  if (!api.GetUniqueId || !api.CommInitRank || !api.AllReduce || !api.Send || !api.Recv || !api.GroupStart || !api.GroupEnd) return nullptr;
  api.lib = lib;
  return &api;
}

struct ShardInfo {
  int rank = 0, own_lo = 0, own_hi = 0;
  std::vector<HaloPiece> recv, send;
  cplx *sendbuf = nullptr, *recvbuf = nullptr;   // NCCL only: [n_rad][sum of piece widths]
};

struct tdde_group {
  std::vector<tdde_handle*> hs;
  std::vector<ShardInfo> info;
  int world = 1;
  void* comm = nullptr;            // ncclComm_t, or nullptr: all shards local
  double** d_bufptr = nullptr;     // device array of the local shards' sum buffers (local all-reduce)
  bool gather = false;             // the in-iteration applies fetch their halo columns themselves (k_apply_mma<GATHER>): no copies for y, z
  cudaStream_t stream = nullptr;
};

// ---- kernels ----
// dst[j * ld_d + lo_d + c] = src[j * ld_s + lo_s + c], c < n, j < n_rad   (halo copy, pack and unpack are all this)
__global__ void k_halo_copy(cplx* __restrict__ dst, int ld_d, int lo_d, const cplx* __restrict__ src, int ld_s, int lo_s, int n, int n_rad) {
  const long long tot = (long long)n * n_rad;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < tot; q += (long long)gridDim.x * blockDim.x) {
    const int j = (int)(q / n), c = (int)(q % n);
    dst[(size_t)j * ld_d + lo_d + c] = src[(size_t)j * ld_s + lo_s + c];
  }
}
// every local buffer <- sum over the local buffers, in shard order (deterministic)
__global__ void k_sum_local(double* const* bufs, int nbuf) {
  const int t = threadIdx.x;
  if (t >= 3) return;
  double s = 0;
  for (int k = 0; k < nbuf; ++k) s += bufs[k][t];
  for (int k = 0; k < nbuf; ++k) bufs[k][t] = s;
}
// the scalar update that the reducing kernel skipped, under the same guard
__global__ void k_finalize(SolverState* st, int fin, int guard, const double* sums) {
  if (guard == 1 && solver_idle(st)) return;
  if (guard == 2 && (st->stalled | (st->status != 0))) return;
  finalize_scalars(st, fin, sums[0], sums[1], sums[2]);
}

// ---- collectives ----
static cplx* shard_vec(tdde_handle* h, int v) { return v == SV_X ? h->X : (v == SV_Y ? h->y : h->z); }

static int copy_grid(long long tot) { return (int)std::max<long long>(1, std::min<long long>((tot + 255) / 256, 4096)); }

// refresh the halo columns of vector v on every local shard
static int group_exchange(tdde_group* g, int v) {
  if (g->gather && v != SV_X) return 0;                      // gathered inside the apply
  cudaStream_t s = g->stream;
  NcclApi* nc = g->comm ? nccl_api() : nullptr;
  if (!g->comm) {
    for (size_t k = 0; k < g->hs.size(); ++k) {
      tdde_handle* h = g->hs[k];
      for (const HaloPiece& pc : g->info[k].recv) {
        tdde_handle* src = nullptr;
        for (size_t q = 0; q < g->hs.size(); ++q) if (g->info[q].rank == pc.peer) src = g->hs[q];
        if (!src) return TDDE_EINVAL;
        k_halo_copy<<<copy_grid((long long)pc.n * h->cfg.n_rad), 256, 0, s>>>(shard_vec(h, v), h->ld, pc.lo, shard_vec(src, v), src->ld, pc.src_lo,
                                                                             pc.n, h->cfg.n_rad);
        h->launches += 1;
      }
    }
    return 0;
  }
  // one shard per process: pack the pieces the neighbours need, exchange them in one NCCL group, unpack the received ones
  tdde_handle* h = g->hs[0];
  ShardInfo& in = g->info[0];
  const int n_rad = h->cfg.n_rad;
  size_t off = 0;
  for (const HaloPiece& pc : in.send) {
    k_halo_copy<<<copy_grid((long long)pc.n * n_rad), 256, 0, s>>>(in.sendbuf + off, pc.n, 0, shard_vec(h, v), h->ld, pc.lo, pc.n, n_rad);
    off += (size_t)pc.n * n_rad;
    h->launches += 1;
  }
  if (nc->GroupStart()) return TDDE_ECUDA;
  off = 0;
  for (const HaloPiece& pc : in.send) {
    if (nc->Send(in.sendbuf + off, (size_t)pc.n * n_rad * 2, kNcclFloat64, pc.peer, g->comm, s)) return TDDE_ECUDA;
    off += (size_t)pc.n * n_rad;
  }
  off = 0;
  for (const HaloPiece& pc : in.recv) {
    if (nc->Recv(in.recvbuf + off, (size_t)pc.n * n_rad * 2, kNcclFloat64, pc.peer, g->comm, s)) return TDDE_ECUDA;
    off += (size_t)pc.n * n_rad;
  }
  if (nc->GroupEnd()) return TDDE_ECUDA;
  off = 0;
  for (const HaloPiece& pc : in.recv) {
    k_halo_copy<<<copy_grid((long long)pc.n * n_rad), 256, 0, s>>>(shard_vec(h, v), h->ld, pc.lo, in.recvbuf + off, pc.n, 0, pc.n, n_rad);
    off += (size_t)pc.n * n_rad;
    h->launches += 1;
  }
  return 0;
}

// the sums every shard's reducing kernel left in shard_sums -> their total on every shard -> the scalar update
static int group_reduce(tdde_group* g, int fin, int guard) {
  cudaStream_t s = g->stream;
  if (g->hs.size() > 1) k_sum_local<<<1, 32, 0, s>>>(g->d_bufptr, (int)g->hs.size());
  if (g->comm) {
    NcclApi* nc = nccl_api();
    if (nc->AllReduce(g->hs[0]->shard_sums, g->hs[0]->shard_sums, 3, kNcclFloat64, kNcclSum, g->comm, s)) return TDDE_ECUDA;
  }
  for (tdde_handle* h : g->hs) { k_finalize<<<1, 1, 0, s>>>(h->d_st, fin, guard, h->shard_sums); h->launches += 1; }
  return 0;
}

// ---- one CN step on all shards in lock step (the phases of enqueue_step_start / enqueue_iteration in tdde_driver.cu) ----
#define EACH(expr) for (tdde_handle* h : g->hs) { int rc_ = (expr); if (rc_) return rc_; }

static int group_step_start(tdde_group* g) {
  const cplx one = make_double2(1.0, 0.0);
  int rc;
  if ((rc = group_exchange(g, SV_X))) return rc;
  EACH(enqueue_apply(h, h->X, h->r, nullptr, BLK_H0, one, true, h->d_g, &h->d_st->step_idx, 2, FIN_RES0, h->d_st, nullptr, 1,
                     make_double2(0.0, -h->cfg.dt), h->rhat));
  if ((rc = group_reduce(g, FIN_RES0, 2))) return rc;
  EACH(enqueue_apply(h, h->X, h->s, h->r, BLK_S, one, false, h->d_zero_g, nullptr, 2, FIN_R0S, h->d_st, nullptr, 2));
  return group_reduce(g, FIN_R0S, 2);
}

static int group_iteration(tdde_group* g) {
  int rc;
  std::vector<char> fused(g->hs.size(), 0);
  size_t k = 0;
  for (tdde_handle* h : g->hs) { bool f = false; if ((rc = enqueue_vec_update(h, 0, h->d_st, &f))) return rc; fused[k++] = f; }   // p-update
  k = 0;
  for (tdde_handle* h : g->hs) { if ((rc = enqueue_precond(h, h->p, h->y, h->d_st, fused[k++] != 0))) return rc; }               // y = M^-1 p
  if ((rc = group_exchange(g, SV_Y))) return rc;
  EACH(enqueue_apply(h, h->y, h->v, h->rhat, BLK_MP, make_double2(0.0, h->tau), true, h->d_g, &h->d_st->step_idx, 1, FIN_ALPHA, h->d_st, h->p));
  if ((rc = group_reduce(g, FIN_ALPHA, 1))) return rc;
  k = 0;
  for (tdde_handle* h : g->hs) { bool f = false; if ((rc = enqueue_vec_update(h, 1, h->d_st, &f))) return rc; fused[k++] = f; }   // s-update, ||s||
  if ((rc = group_reduce(g, FIN_S, 1))) return rc;
  for (tdde_handle* h : g->hs) h->launches += launch_vec_halfexit(make_vec_args(h, h->d_st, FIN_NONE), g->stream);
  k = 0;
  for (tdde_handle* h : g->hs) { if ((rc = enqueue_precond(h, h->s, h->z, h->d_st, fused[k++] != 0))) return rc; }               // z = M^-1 s
  if ((rc = group_exchange(g, SV_Z))) return rc;
  EACH(enqueue_apply(h, h->z, h->t, h->s, BLK_MP, make_double2(0.0, h->tau), true, h->d_g, &h->d_st->step_idx, 1, FIN_OMEGA, h->d_st, h->s));
  if ((rc = group_reduce(g, FIN_OMEGA, 1))) return rc;
  for (tdde_handle* h : g->hs) h->launches += launch_vec_xr(make_vec_args(h, h->d_st, FIN_R), g->stream);
  return group_reduce(g, FIN_R, 1);
}

static int group_step(tdde_group* g, int n_iter) {
  int rc;
  if ((rc = group_step_start(g))) return rc;
  for (int it = 0; it < n_iter; ++it)
    if ((rc = group_iteration(g))) return rc;
  for (tdde_handle* h : g->hs) h->launches += launch_step_close(h->d_st, g->stream);
  return 0;
}

// ---- C ABI ----
extern "C" int tdde_nccl_unique_id(void* id128) {
  if (!id128) return TDDE_EINVAL;
  NcclApi* nc = nccl_api();
  if (!nc) { g_last_cuda_error = "libnccl.so.2 could not be loaded"; return TDDE_ECUDA; }
  NcclId id;
  if (nc->GetUniqueId(&id)) { g_last_cuda_error = "ncclGetUniqueId failed"; return TDDE_ECUDA; }
  std::memcpy(id128, &id, sizeof(id));
  return 0;
}

extern "C" void tdde_group_destroy(tdde_group* g) {
  if (!g) return;
  for (size_t k = 0; k < g->hs.size(); ++k) {
    tdde_handle* h = g->hs[k];
    if (h->shard_sums) cudaFree(h->shard_sums);
    h->shard_sums = nullptr; h->own_lo = 0; h->own_hi = 0; h->nbrL = h->nbrR = nullptr; h->shiftL = h->shiftR = 0;
    if (g->info[k].sendbuf) cudaFree(g->info[k].sendbuf);
    if (g->info[k].recvbuf) cudaFree(g->info[k].recvbuf);
  }
  if (g->d_bufptr) cudaFree(g->d_bufptr);
  if (g->comm) { NcclApi* nc = nccl_api(); if (nc && nc->CommDestroy) nc->CommDestroy(g->comm); }
  cudaGetLastError();
  delete g;
}

extern "C" int tdde_group_create(tdde_group** out, int32_t n_local, tdde_handle* const* handles, const tdde_shard* shards, const void* nccl_id128) {
  if (!out) return TDDE_EINVAL;
  *out = nullptr;
  if (n_local < 1 || !handles || !shards) return TDDE_EINVAL;
  if (nccl_id128 && n_local != 1) return TDDE_EINVAL;                      // one shard per process with NCCL
  const int world = shards[0].world;
  if (!nccl_id128 && world != n_local) return TDDE_EINVAL;                 // without NCCL every shard of the job must be local
  tdde_handle* h0 = handles[0];
  if (!h0) return TDDE_EINVAL;
  DeviceGuard dg(h0->device);
  tdde_group* g = new (std::nothrow) tdde_group;
  if (!g) return TDDE_ENOMEM;
  g->world = world; g->stream = h0->stream;
  auto fail = [&](int rc) { tdde_group_destroy(g); return rc; };
  for (int k = 0; k < n_local; ++k) {
    tdde_handle* h = handles[k];
    const tdde_shard& sd = shards[k];
    if (!h || h->shard_sums || h->device != h0->device || h->stream != h0->stream) return fail(TDDE_EINVAL);
    if (h->cfg.n_rad != h0->cfg.n_rad || h->user_terms != h0->user_terms || h->cfg.dt != h0->cfg.dt || h->cfg.rtol != h0->cfg.rtol ||
        h->cfg.max_iter != h0->cfg.max_iter || sd.world != world || sd.rank < 0 || sd.rank >= world)
      return fail(TDDE_EINVAL);
    if (sd.own_lo < 0 || sd.own_hi > h->cfg.n_ang || sd.own_lo >= sd.own_hi || sd.n_recv < 0 || sd.n_send < 0) return fail(TDDE_EINVAL);
    ShardInfo in;
    in.rank = sd.rank; in.own_lo = sd.own_lo; in.own_hi = sd.own_hi;
    size_t nrecv = 0, nsend = 0;
    for (int q = 0; q < sd.n_recv; ++q) {
      HaloPiece pc{sd.recv_rank[q], sd.recv_lo[q], sd.recv_src_lo[q], sd.recv_n[q]};
      // a halo piece lies outside the owned slab and inside the local channels
      if (pc.n <= 0 || pc.lo < 0 || pc.lo + pc.n > h->cfg.n_ang || (pc.lo < sd.own_hi && pc.lo + pc.n > sd.own_lo) || pc.peer < 0 ||
          pc.peer >= world || pc.peer == sd.rank || pc.src_lo < 0)
        return fail(TDDE_EINVAL);
      in.recv.push_back(pc); nrecv += pc.n;
    }
    for (int q = 0; q < sd.n_send; ++q) {
      HaloPiece pc{sd.send_rank[q], sd.send_lo[q], 0, sd.send_n[q]};
      if (pc.n <= 0 || pc.lo < sd.own_lo || pc.lo + pc.n > sd.own_hi || pc.peer < 0 || pc.peer >= world || pc.peer == sd.rank) return fail(TDDE_EINVAL);
      in.send.push_back(pc); nsend += pc.n;
    }
    g->hs.push_back(h);
    g->info.push_back(in);
    ShardInfo& inf = g->info.back();
    if (cudaMalloc((void**)&h->shard_sums, 4 * sizeof(double)) != cudaSuccess) { h->shard_sums = nullptr; return fail(TDDE_ENOMEM); }
    cudaMemsetAsync(h->shard_sums, 0, 4 * sizeof(double), g->stream);
    h->own_lo = sd.own_lo; h->own_hi = sd.own_hi;
    // halo columns of every work vector must be exactly zero (see the header): clear them all
    cplx* vecs[] = {h->X, h->r, h->rhat, h->p, h->v, h->s, h->t, h->y, h->z};
    for (cplx* v : vecs) cudaMemsetAsync(v, 0, (size_t)h->nint * sizeof(cplx), g->stream);
    if (nccl_id128) {
      if (nsend && cudaMalloc((void**)&inf.sendbuf, nsend * h->cfg.n_rad * sizeof(cplx)) != cudaSuccess) return fail(TDDE_ENOMEM);
      if (nrecv && cudaMalloc((void**)&inf.recvbuf, nrecv * h->cfg.n_rad * sizeof(cplx)) != cudaSuccess) return fail(TDDE_ENOMEM);
    }
  }
  // local pieces must name a local owner whose owned slab covers them
  if (!nccl_id128) {
    for (size_t k = 0; k < g->hs.size(); ++k)
      for (const HaloPiece& pc : g->info[k].recv) {
        bool ok = false;
        for (size_t q = 0; q < g->hs.size(); ++q)
          if (g->info[q].rank == pc.peer && pc.src_lo >= g->info[q].own_lo && pc.src_lo + pc.n <= g->info[q].own_hi) ok = true;
        if (!ok) return fail(TDDE_EINVAL);
      }
    // Fused gather: every shard runs k_apply_mma in the iteration and has at most one neighbour per side that owns its whole halo
    bool gather = !std::getenv("TDDE_NO_GATHER") && g->hs.size() > 1;
    for (size_t k = 0; k < g->hs.size() && gather; ++k) {
      tdde_handle* h = g->hs[k];
      const ShardInfo& in = g->info[k];
      if (h->path != 1 || h->seg_len_m <= 0 || !h->use_subst || h->cfg.n_terms == 0 || in.recv.size() > 2) gather = false;
      int nl = 0, nr = 0;
      for (const HaloPiece& pc : in.recv) {
        if (pc.lo == 0 && pc.n == in.own_lo) ++nl;
        else if (pc.lo == in.own_hi && pc.lo + pc.n == h->cfg.n_ang) ++nr;
        else gather = false;
      }
      if (nl > 1 || nr > 1) gather = false;
    }
    if (gather) {
      for (size_t k = 0; k < g->hs.size(); ++k)
        for (const HaloPiece& pc : g->info[k].recv) {
          tdde_handle* src = nullptr;
          for (size_t q = 0; q < g->hs.size(); ++q) if (g->info[q].rank == pc.peer) src = g->hs[q];
          if (pc.lo == 0) { g->hs[k]->nbrL = src; g->hs[k]->shiftL = pc.src_lo - pc.lo; }
          else { g->hs[k]->nbrR = src; g->hs[k]->shiftR = pc.src_lo - pc.lo; }
        }
      g->gather = true;
    }
    std::vector<double*> ptrs;
    for (tdde_handle* h : g->hs) ptrs.push_back(h->shard_sums);
    if (cudaMalloc((void**)&g->d_bufptr, ptrs.size() * sizeof(double*)) != cudaSuccess) return fail(TDDE_ENOMEM);
    cudaMemcpyAsync(g->d_bufptr, ptrs.data(), ptrs.size() * sizeof(double*), cudaMemcpyHostToDevice, g->stream);
    cudaStreamSynchronize(g->stream);
  } else {
    NcclApi* nc = nccl_api();
    if (!nc) { g_last_cuda_error = "libnccl.so.2 could not be loaded"; return fail(TDDE_ECUDA); }
    NcclId id;
    std::memcpy(&id, nccl_id128, sizeof(id));
    if (nc->CommInitRank(&g->comm, world, id, shards[0].rank)) { g->comm = nullptr; g_last_cuda_error = "ncclCommInitRank failed"; return fail(TDDE_ECUDA); }
  }
  if (cudaStreamSynchronize(g->stream) != cudaSuccess) return fail(tdde_cuda_fail(cudaGetLastError(), "tdde_group_create"));
  *out = g;
  return 0;
}

extern "C" int tdde_group_propagate(tdde_group* g, tdde_c64* const* c_dev, int64_t n_steps, const double* g_table, tdde_stats* st) {
  if (!g || !c_dev || n_steps < 0 || g->hs.empty()) return TDDE_EINVAL;
  tdde_handle* h0 = g->hs[0];
  if (n_steps > 0 && h0->user_terms > 0 && !g_table) return TDDE_EINVAL;
  for (size_t k = 0; k < g->hs.size(); ++k) if (!c_dev[k]) return TDDE_EINVAL;
  DeviceGuard dg(h0->device);
  if (st) std::memset(st, 0, sizeof(*st));
  if (n_steps == 0) return 0;
  int rc;
  int nspec = 1;
  for (size_t k = 0; k < g->hs.size(); ++k) {
    tdde_handle* h = g->hs[k];
    std::vector<double> gbuf;
    const double* gt = map_g(h, g_table, n_steps, gbuf);
    if ((rc = upload_g(h, gt, n_steps))) return rc;
    CU(cudaStreamSynchronize(h->stream));                  // gbuf is about to go out of scope
    h->h_st->status = 0; h->h_st->stalled = 0; h->h_st->done = 1; h->h_st->force = 0;
    h->h_st->rtol2 = h->cfg.rtol * h->cfg.rtol; h->h_st->max_half = 2 * h->cfg.max_iter;
    CU(cudaMemcpyAsync(h->d_st, h->h_st, sizeof(SolverState), cudaMemcpyHostToDevice, h->stream));
    h->launches += launch_to_internal(reinterpret_cast<const cplx*>(c_dev[k]), h->X, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
    h->launches += launch_step_open(h->d_st, 0, 0, 0, h->stream);
    nspec = std::max(nspec, h->nspec);
  }
  rc = 0;
  for (long long step = 0; step < n_steps && !rc; ++step) {
    if ((rc = group_step(g, nspec))) break;
    if ((rc = sync_state(h0))) break;                      // one host read per step; every shard holds the same scalars
    if (h0->h_st->status != 0) { rc = h0->h_st->status; break; }
    while (h0->h_st->stalled) {
      for (tdde_handle* h : g->hs) h->launches += launch_step_open(h->d_st, 0, 0, 1, g->stream);
      const int more = std::max(2, nspec);
      for (int it = 0; it < more && !rc; ++it) rc = group_iteration(g);
      if (rc) break;
      for (tdde_handle* h : g->hs) h->launches += launch_step_close(h->d_st, g->stream);
      if ((rc = sync_state(h0))) break;
      if (h0->h_st->status != 0) { rc = h0->h_st->status; break; }
      if (!h0->h_st->stalled) nspec = std::min(h0->cfg.max_iter, std::max(nspec, (h0->h_st->last_half_iters + 1) / 2));
    }
  }
  for (size_t k = 0; k < g->hs.size(); ++k) {
    tdde_handle* h = g->hs[k];
    h->nspec = nspec;
    h->launches += launch_to_boundary(h->X, reinterpret_cast<cplx*>(c_dev[k]), h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  }
  CU(cudaStreamSynchronize(g->stream));
  fill_stats(h0, st);
  CU(cudaGetLastError());
  return rc;
}
