// tdde_misc.cu -- measurement helpers and small exports of tdde.h.
#include <cstring>
#include "tdde_handle.h"

extern "C" const char* tdde_strerror(int status) {
  switch (status) {
    case TDDE_OK: return "ok";
    case TDDE_EINVAL: return "invalid argument";
    case TDDE_ENOMEM: return "out of memory";
    case TDDE_ECUDA: return "CUDA error (see tdde_last_cuda_error)";
    case TDDE_ESINGULAR: return "singular block in the preconditioner LU";
    case TDDE_EBREAKDOWN: return "BiCGSTAB breakdown";
    case TDDE_ENOCONV: return "BiCGSTAB did not converge within max_iter";
    default: return "unknown status";
  }
}

extern "C" const char* tdde_last_cuda_error(void) { return g_last_cuda_error.c_str(); }
extern "C" int tdde_version(void) { return 1; }
extern "C" int64_t tdde_launch_count(const tdde_handle* h) { return h ? h->launches : 0; }
extern "C" int tdde_apply_path(const tdde_handle* h) { return h ? h->path : -1; }

extern "C" int tdde_time_kernel(tdde_handle* h, int32_t which, int32_t reps, const double* g, double* ms_out) {
  if (!h || !ms_out || reps <= 0 || which < 0 || which > 6) return TDDE_EINVAL;
  if (which == 0 && h->cfg.n_terms > 0 && !g) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  cudaStream_t s = h->stream;
  SolverState* sb = h->d_st_bench;
  // finite, non-trivial data in every work vector
  cplx* vecs[] = {h->X, h->r, h->rhat, h->p, h->v, h->s, h->t, h->y, h->z};
  unsigned seed = 1;
  for (cplx* v : vecs) h->launches += launch_fill(v, h->nint, seed++, s);
  if (h->cfg.n_terms > 0 && g)
    CU(cudaMemcpyAsync(h->d_g_small, g, h->cfg.n_terms * sizeof(double), cudaMemcpyHostToDevice, s));
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  const cplx itau = make_double2(0.0, h->tau);
  int rc = 0;
  auto once = [&]() -> int {
    switch (which) {
      case 0: return enqueue_apply(h, h->y, h->v, h->rhat, BLK_MP, itau, true, h->d_g_small, nullptr, 0, FIN_ALPHA, sb, h->p);   // as the iteration runs it
      case 1: return enqueue_precond(h, h->p, h->y, nullptr);
      case 2: h->launches += launch_vec_p(make_vec_args(h, sb, FIN_NONE), s); return 0;
      case 3: h->launches += launch_vec_s(make_vec_args(h, sb, FIN_NONE), s); return 0;
      case 4: h->launches += launch_vec_xr(make_vec_args(h, sb, FIN_NONE), s); return 0;
      case 5: h->launches += launch_to_internal(h->z, h->t, h->cfg.n_ang, h->cfg.n_rad, h->ld, s); return 0;
      default: return enqueue_apply(h, h->y, h->z, h->y, BLK_S, make_double2(0, 0), false, h->d_zero_g, nullptr, 0, FIN_NONE, sb);
    }
  };
  for (int w = 0; w < 3 && !rc; ++w) rc = once();
  if (!rc) {
    CU(cudaEventRecord(e0, s));
    for (int r = 0; r < reps && !rc; ++r) rc = once();
    CU(cudaEventRecord(e1, s));
    CU(cudaEventSynchronize(e1));
    float ms = 0;
    CU(cudaEventElapsedTime(&ms, e0, e1));
    *ms_out = (double)ms / reps;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  CU(cudaGetLastError());
  return rc;
}

extern "C" int tdde_fp64_peak(void* cuda_stream, double* flops_out) {
  if (!flops_out) return TDDE_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double* d = nullptr;
  CU(cudaMalloc((void**)&d, sizeof(double)));
  const int blocks = tdde_num_sms() * 8, threads = 256, iters = 4096;
  launch_dfma_peak(d, blocks, threads, 64, s);
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  CU(cudaEventRecord(e0, s));
  launch_dfma_peak(d, blocks, threads, iters, s);
  CU(cudaEventRecord(e1, s));
  CU(cudaEventSynchronize(e1));
  float ms = 0;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  const double fmas = (double)blocks * threads * (double)iters * 64.0;   // 8 chains x 8 unrolled
  *flops_out = 2.0 * fmas / (ms * 1e-3);
  CU(cudaGetLastError());
  return 0;
}
