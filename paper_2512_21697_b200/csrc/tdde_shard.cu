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
#include <cstring>
#include <vector>
#include <dlfcn.h>
#include "tdde_handle.h"
#include "tdde_reduce.cuh"

enum ShardVec { SV_X = 0, SV_Y = 1, SV_Z = 2 };

struct HaloPiece { int peer, lo, src_lo, n; };   // recv: [lo, lo+n) here = [src_lo, ..) on peer; send: [lo, lo+n) here goes to peer

// ---- NCCL through dlopen (torch ships libnccl.so.2; no link-time dependency, the single-GPU library never needs it) ----
struct NcclApi {
  void* lib = nullptr;
  int (*GetUniqueId)(void*) = nullptr;
  int (*CommInitRank)(void**, int, struct NcclId, int) = nullptr;
  int (*AllReduce)(const void*, void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*Send)(const void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*Recv)(void*, size_t, int, int, void*, cudaStream_t) = nullptr;
  int (*GroupStart)() = nullptr;
  int (*GroupEnd)() = nullptr;
  int (*CommDestroy)(void*) = nullptr;
};
struct NcclId { char bytes[128]; };
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
