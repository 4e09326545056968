// tdde_misc.cu -- measurement helpers and small exports of tdde.h.
#include <cstring>
#include <vector>
#include "tdde_handle.h"
#include "tdde_reduce.cuh"

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
extern "C" int tdde_version(void) { return 2; }
extern "C" int tdde_apply_path(const tdde_handle* h) { return h ? h->path : -1; }
#ifdef TDDE_WITH_BENCH
extern "C" int tdde_iter_apply_kernel(const tdde_handle* h) {
  if (!h) return -1;
  return (h->path == 1 && h->use_subst && h->cfg.n_terms > 0 && h->seg_len_m > 0) ? 3 : h->path;
}
#endif

#ifdef TDDE_WITH_BENCH
extern "C" int64_t tdde_launch_count(const tdde_handle* h) { return h ? h->launches : 0; }

extern "C" int tdde_time_kernel(tdde_handle* h, int32_t which, int32_t reps, const double* g, double* ms_out) {
  if (!h || !ms_out || reps <= 0 || which < 0 || which > 6) return TDDE_EINVAL;
  if (which == 0 && h->user_terms > 0 && !g) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  std::vector<double> gbuf;
  g = map_g(h, g, 1, gbuf);
  cudaStream_t s = h->stream;
  SolverState* sb = h->d_st_bench;
  // finite, non-trivial data in every work vector
  cplx* vecs[] = {h->X, h->r, h->rhat, h->p, h->v, h->s, h->t, h->y, h->z};
  unsigned seed = 1;
  for (cplx* v : vecs) h->launches += launch_fill(v, h->nint, seed++, s);
  if (h->cfg.n_terms > 0 && g)
    CU(cudaMemcpyAsync(h->d_g_small, g, h->cfg.n_terms * sizeof(double), cudaMemcpyHostToDevice, s));
  ScopedEvent e0, e1;
  CU(e0.create());
  CU(e1.create());
  const cplx itau = make_double2(0.0, h->tau);
  int rc = 0;
  bool fused_avail = false, fused_tmp = false;
  if (which == 1) {                                 // does the fused update exist for this problem?  (also fills rsm / rsp)
    if ((rc = enqueue_vec_update(h, 0, sb, &fused_avail))) return rc;
  }
  auto once = [&]() -> int {
    switch (which) {
      case 0: return enqueue_apply(h, h->y, h->v, h->rhat, BLK_MP, itau, true, h->d_g_small, nullptr, 0, FIN_ALPHA, sb, h->p);   // as the iteration runs it
      // 1-3 as an iteration runs them: the p- and s-updates carry the spike products of the solve that follows (when available),
      // and the solve then starts at its Schur step
      case 1: return enqueue_precond(h, h->p, h->y, nullptr, fused_avail);
      case 2: return enqueue_vec_update(h, 0, sb, &fused_tmp);
      case 3: return enqueue_vec_update(h, 1, sb, &fused_tmp);
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
  CU(cudaGetLastError());
  return rc;
}

extern "C" int tdde_apply_coupling(tdde_handle* h, tdde_c64 beta, const double* g, const tdde_c64* x_dev, const tdde_c64* addv_dev,
                                   const tdde_c64* aux_dev, tdde_c64* y_dev, int32_t which, double* dots) {
  if (!h || !g || !x_dev || !addv_dev || !y_dev || y_dev == x_dev || y_dev == addv_dev || y_dev == aux_dev) return TDDE_EINVAL;
  if (h->path != 1 || h->cfg.n_terms == 0 || !h->use_subst) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  std::vector<double> gbuf;
  g = map_g(h, g, 1, gbuf);
  cudaStream_t s = h->stream;
  CU(cudaMemcpyAsync(h->d_g_small, g, h->cfg.n_terms * sizeof(double), cudaMemcpyHostToDevice, s));
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(x_dev), h->y, h->cfg.n_ang, h->cfg.n_rad, h->ld, s);
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(addv_dev), h->p, h->cfg.n_ang, h->cfg.n_rad, h->ld, s);
  if (aux_dev) h->launches += launch_to_internal(reinterpret_cast<const cplx*>(aux_dev), h->rhat, h->cfg.n_ang, h->cfg.n_rad, h->ld, s);
  // FIN_DOTS parks the raw sums in the (never-idle) bench state
  const int keep = h->seg_len_m;
  if (which == 1) h->seg_len_m = 0;
  SolverState* sb = h->d_st_bench;
  int rc = enqueue_apply(h, h->y, h->v, aux_dev ? h->rhat : nullptr, BLK_MP, make_double2(beta.re, beta.im), true, h->d_g_small, nullptr, 0,
                         FIN_DOTS, sb, h->p);
  h->seg_len_m = keep;
  if (rc) return rc;
  h->launches += launch_to_boundary(h->v, reinterpret_cast<cplx*>(y_dev), h->cfg.n_ang, h->cfg.n_rad, h->ld, s);
  SolverState hs;
  CU(cudaMemcpyAsync(&hs, sb, sizeof(SolverState), cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  if (dots) { dots[0] = hs.rho_old.x; dots[1] = hs.rho_old.y; dots[2] = hs.res2; }
  CU(cudaGetLastError());
  return 0;
}

extern "C" int tdde_fp64_peak(void* cuda_stream, double* flops_out) {
  if (!flops_out) return TDDE_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double* d = nullptr;
  CU(cudaMalloc((void**)&d, sizeof(double)));
  const int blocks = tdde_num_sms() * 8, threads = 256, iters = 4096;
  launch_dfma_peak(d, blocks, threads, 64, s);
  ScopedEvent e0, e1;
  CU(e0.create());
  CU(e1.create());
  CU(cudaEventRecord(e0, s));
  launch_dfma_peak(d, blocks, threads, iters, s);
  CU(cudaEventRecord(e1, s));
  CU(cudaEventSynchronize(e1));
  float ms = 0;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaFree(d);
  const double fmas = (double)blocks * threads * (double)iters * 64.0;   // 8 chains x 8 unrolled
  *flops_out = 2.0 * fmas / (ms * 1e-3);
  CU(cudaGetLastError());
  return 0;
}

// mode 0: DFMA only (= tdde_fp64_peak), 1: DMMA only, 2: DMMA and DFMA mixed in one warp (8 : 32, the mix of k_apply_mma)
extern "C" int tdde_fp64_pipe_probe(void* cuda_stream, int32_t mode, double* flops_out) {
  if (!flops_out || mode < 0 || mode > 2) return TDDE_EINVAL;
  if (mode == 0) return tdde_fp64_peak(cuda_stream, flops_out);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double* d = nullptr;
  CU(cudaMalloc((void**)&d, sizeof(double)));
  const int blocks = tdde_num_sms() * 2, threads = 256, iters = 20000;
  launch_fp64_pipe_probe(d, blocks, threads, 64, mode, s);
  ScopedEvent e0, e1;
  CU(e0.create());
  CU(e1.create());
  CU(cudaEventRecord(e0, s));
  launch_fp64_pipe_probe(d, blocks, threads, iters, mode, s);
  CU(cudaEventRecord(e1, s));
  CU(cudaEventSynchronize(e1));
  float ms = 0;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  cudaFree(d);
  const double warps = (double)blocks * threads / 32.0;
  const double flop_per_iter = 8 * 2.0 * 256.0 + (mode == 2 ? 32 * 2.0 * 32.0 : 0.0);      // per warp
  *flops_out = warps * (double)iters * flop_per_iter / (ms * 1e-3);
  CU(cudaGetLastError());
  return 0;
}
#endif  // TDDE_WITH_BENCH

// ---- observables (Eq. 33) ----
// P[a][e] = |sum_j conj(V_k(a)[j][e]) u[j][a]|^2 with u = S c in the internal layout.  Thread = channel (coalesced reads of u),
// PJ_NE states per thread; the eigenvector entries of a row are contiguous in e and (per kappa-class) warp-uniform.
#define PJ_NE 8
__global__ void __launch_bounds__(128) k_project(const cplx* __restrict__ u, const cplx* __restrict__ V, const int* __restrict__ cls,
                                                  double* __restrict__ P, int n_ang, int n_rad, int ld, int n_states) {
  const int a = blockIdx.x * 128 + threadIdx.x;
  if (a >= n_ang) return;
  const int e0 = blockIdx.y * PJ_NE;
  const cplx* Vk = V + (size_t)cls[a] * n_rad * n_states + e0;
  const int ne = min(PJ_NE, n_states - e0);
  cplx acc[PJ_NE];
#pragma unroll
  for (int e = 0; e < PJ_NE; ++e) acc[e] = make_double2(0, 0);
  for (int j = 0; j < n_rad; ++j) {
    const cplx uj = u[(size_t)j * ld + a];
    const cplx* vr = Vk + (size_t)j * n_states;
#pragma unroll
    for (int e = 0; e < PJ_NE; ++e)
      if (e < ne) cfma_conj(acc[e], __ldg(vr + e), uj);
  }
  for (int e = 0; e < ne; ++e) P[(size_t)a * n_states + e0 + e] = acc[e].x * acc[e].x + acc[e].y * acc[e].y;
}

extern "C" int tdde_set_eigenstates(tdde_handle* h, int32_t n_states, const tdde_c64* V) {
  if (!h || n_states <= 0 || !V) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  const int n_cls = h->cfg.n_cls, n_rad = h->cfg.n_rad;
  CU(cudaStreamSynchronize(h->stream));
  if (h->d_eig) { cudaFree(h->d_eig); h->d_eig = nullptr; }
  if (h->d_proj) { cudaFree(h->d_proj); h->d_proj = nullptr; }
  h->n_states = 0;
  // [k][e][j] at the boundary -> [k][j][e] on the device (the kernel walks j and wants the states of a row contiguous)
  std::vector<zc> T((size_t)n_cls * n_rad * n_states);
  const zc* Vh = reinterpret_cast<const zc*>(V);
  for (int k = 0; k < n_cls; ++k)
    for (int e = 0; e < n_states; ++e)
      for (int j = 0; j < n_rad; ++j) T[((size_t)k * n_rad + j) * n_states + e] = Vh[((size_t)k * n_states + e) * n_rad + j];
  CU(cudaMalloc((void**)&h->d_eig, T.size() * sizeof(cplx)));
  CU(cudaMemcpy(h->d_eig, T.data(), T.size() * sizeof(cplx), cudaMemcpyHostToDevice));
  CU(cudaMalloc((void**)&h->d_proj, (size_t)h->cfg.n_ang * n_states * sizeof(double)));
  h->n_states = n_states;
  return 0;
}

extern "C" int tdde_project(tdde_handle* h, const tdde_c64* c_dev, double* P_host) {
  if (!h || !c_dev || !P_host || h->n_states <= 0) return TDDE_EINVAL;
  DeviceGuard dg(h->device);
  int rc;
  h->launches += launch_to_internal(reinterpret_cast<const cplx*>(c_dev), h->y, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->stream);
  // u = S c: the S-only operator apply (beta = 0), no fused reduction
  if ((rc = enqueue_apply(h, h->y, h->z, nullptr, BLK_S, make_double2(0, 0), false, h->d_zero_g, nullptr, 0, FIN_NONE, h->d_st))) return rc;
  dim3 grid((h->cfg.n_ang + 127) / 128, (h->n_states + PJ_NE - 1) / PJ_NE);
  k_project<<<grid, 128, 0, h->stream>>>(h->z, h->d_eig, h->d_cls, h->d_proj, h->cfg.n_ang, h->cfg.n_rad, h->ld, h->n_states);
  h->launches += 1;
  CU(cudaMemcpyAsync(P_host, h->d_proj, (size_t)h->cfg.n_ang * h->n_states * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CU(cudaStreamSynchronize(h->stream));
  CU(cudaGetLastError());
  return 0;
}
