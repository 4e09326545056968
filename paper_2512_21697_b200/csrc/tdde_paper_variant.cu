#ifdef TDDE_WITH_BENCH
// tdde_paper_variant.cu -- the paper's own formulation on the same GPU, as a comparator:
//   * the global matrix A(t) = S + i dt/2 H(t) is held in CSR, structure allocated once;
//   * an assembly kernel recomputes every non-zero from the stored radial matrices and angular couplings each step,
//     consecutive threads writing consecutive entries of a CSR row (Eq. 17);
//   * y = A x is a CSR SpMV (the paper calls cuSPARSE / rocSPARSE); here a warp-per-row kernel.
// It is NOT on the product path: tdde_paper_variant() exists so that bench.py and the tests can time and check it
// beside the matrix-free apply.  Vectors are in the boundary layout (global index I = a * n_rad + i), as in the paper.
// Only problems on the banded path are supported (the non-zero pattern is then band (x) band, known in closed form).
#include <vector>
#include "tdde_handle.h"
#include "tdde_reduce.cuh"

struct PvArgs {
  int n_ang, n_rad, ld, w, T, MM;            // MM = largest channel offset
  const int* cls;
  const cplx* Mcol;                          // [n_cls][n_rad][2w+1] column-band of M+ = S + i tau H0
  const cplx* Rall;                          // [n_rad][T][2w+1]
  const cplx* Aoff;                          // [n_slots][ld]
  int m[TDDE_MAX_TERMS], slot0[TDDE_MAX_TERMS];
  double gtau[TDDE_MAX_TERMS];               // tau * g_L
  const long long* chan_base;                // [n_ang]   first non-zero of channel a' (row i = 0)
  const int* nch;                            // [n_ang]   coupled channels of a'
  const int* rad_pref;                       // [n_rad+1] prefix of per-row radial widths
  long long* rowptr;                         // [n + 1]
  int* col;                                  // [nnz]
  cplx* val;                                 // [nnz]
};

__device__ __forceinline__ long long pv_row_start(const PvArgs& p, int a, int i) {
  return p.chan_base[a] + (long long)p.nch[a] * p.rad_pref[i];
}

__global__ void k_pv_rowptr(PvArgs p, long long n, long long nnz) {
  for (long long I = (long long)blockIdx.x * blockDim.x + threadIdx.x; I <= n; I += (long long)gridDim.x * blockDim.x) {
    if (I == n) { p.rowptr[I] = nnz; continue; }
    p.rowptr[I] = pv_row_start(p, (int)(I / p.n_rad), (int)(I % p.n_rad));
  }
}

// one warp per CSR row; MODE 0: column indices (once), MODE 1: values (every step)
template <int MODE>
__global__ void __launch_bounds__(256) k_pv_assemble(PvArgs p, long long n) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  const int nd = 2 * p.w + 1;
  for (long long I = warp0; I < n; I += nwarps) {
    const int a1 = (int)(I / p.n_rad), i = (int)(I % p.n_rad);
    const int alo = max(a1 - p.MM, 0), jlo = max(i - p.w, 0);
    const int nr = p.rad_pref[i + 1] - p.rad_pref[i], len = p.nch[a1] * nr;
    const long long base = pv_row_start(p, a1, i);
    for (int e = lane; e < len; e += 32) {
      const int a = alo + e / nr, j = jlo + e % nr;
      if (MODE == 0) { p.col[base + e] = a * p.n_rad + j; continue; }
      const int eb = i - j + p.w;                                     // column-band position of (i, j)
      cplx v = make_double2(0, 0);
      if (a == a1) v = p.Mcol[((size_t)p.cls[a1] * p.n_rad + j) * nd + eb];
      const int o = a - a1, ao = o < 0 ? -o : o;
      if (o != 0) {
        for (int L = 0; L < p.T; ++L) {
          if (p.m[L] < ao) continue;
          const int q = o < 0 ? o + p.m[L] : p.m[L] + o - 1;
          const cplx A = p.Aoff[(size_t)(p.slot0[L] + q) * p.ld + a1];
          const cplx R = p.Rall[((size_t)j * p.T + L) * nd + eb];
          const cplx ar = cmul(A, R);
          v.x -= p.gtau[L] * ar.y;                                    // += i * tau g_L * (A R)
          v.y += p.gtau[L] * ar.x;
        }
      }
      p.val[base + e] = v;
    }
  }
}

__global__ void __launch_bounds__(256) k_pv_spmv(PvArgs p, long long n, const cplx* __restrict__ x, cplx* __restrict__ y) {
  const int lane = threadIdx.x & 31;
  const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
  for (long long I = warp0; I < n; I += nwarps) {
    const long long b = p.rowptr[I], e1 = p.rowptr[I + 1];
    cplx acc = make_double2(0, 0);
    for (long long e = b + lane; e < e1; e += 32) cfma(acc, p.val[e], x[p.col[e]]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      acc.x += __shfl_down_sync(0xffffffffu, acc.x, o);
      acc.y += __shfl_down_sync(0xffffffffu, acc.y, o);
    }
    if (lane == 0) y[I] = acc;
  }
}

extern "C" int tdde_paper_variant(tdde_handle* h, const double* g, const tdde_c64* x_dev, tdde_c64* y_dev, int32_t reps,
                                  double* ms_assemble, double* ms_spmv, int64_t* nnz_out) {
  if (!h || !x_dev || !y_dev || reps <= 0 || (h->user_terms > 0 && !g)) return TDDE_EINVAL;
  if (h->bW != h->cfg.w0 || !h->g_identity) return TDDE_EINVAL;      // only for problems that ARE an instantiated shape (no zero-filled slots)
  if (h->path != 1) return TDDE_EINVAL;                               // pattern known in closed form only there
  const int n_ang = h->cfg.n_ang, n_rad = h->cfg.n_rad, w = h->cfg.w0, T = h->cfg.n_terms;
  PvArgs p;
  p.n_ang = n_ang; p.n_rad = n_rad; p.ld = h->ld; p.w = w; p.T = T; p.MM = 0;
  p.cls = h->d_cls; p.Mcol = h->d_Mp; p.Rall = h->d_Rall; p.Aoff = h->d_Aoff;
  int s0 = 0;
  for (int L = 0; L < T; ++L) {
    p.m[L] = h->bM0 + h->bMS * L; p.slot0[L] = s0; s0 += 2 * p.m[L];
    p.gtau[L] = h->tau * g[L];
    p.MM = std::max(p.MM, p.m[L]);
  }
  std::vector<long long> chan_base(n_ang);
  std::vector<int> nch(n_ang), rad_pref(n_rad + 1, 0);
  for (int i = 0; i < n_rad; ++i) rad_pref[i + 1] = rad_pref[i] + (std::min(i + w, n_rad - 1) - std::max(i - w, 0) + 1);
  long long nnz = 0;
  for (int a = 0; a < n_ang; ++a) {
    nch[a] = std::min(a + p.MM, n_ang - 1) - std::max(a - p.MM, 0) + 1;
    chan_base[a] = nnz;
    nnz += (long long)nch[a] * rad_pref[n_rad];
  }
  if (nnz_out) *nnz_out = nnz;
  const long long n = h->n;
  long long* d_base = nullptr; int *d_nch = nullptr, *d_pref = nullptr;
  cudaStream_t s = h->stream;
  int rc = 0;
  auto cleanup = [&]() {
    cudaFree(d_base); cudaFree(d_nch); cudaFree(d_pref); cudaFree(p.rowptr); cudaFree(p.col); cudaFree(p.val);
  };
  p.rowptr = nullptr; p.col = nullptr; p.val = nullptr;
#define PV(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = tdde_cuda_fail(e__, #call); cleanup(); return rc; } } while (0)
  PV(cudaMalloc((void**)&d_base, n_ang * sizeof(long long)));
  PV(cudaMalloc((void**)&d_nch, n_ang * sizeof(int)));
  PV(cudaMalloc((void**)&d_pref, (n_rad + 1) * sizeof(int)));
  PV(cudaMalloc((void**)&p.rowptr, (n + 1) * sizeof(long long)));
  PV(cudaMalloc((void**)&p.col, (size_t)nnz * sizeof(int)));
  PV(cudaMalloc((void**)&p.val, (size_t)nnz * sizeof(cplx)));
  PV(cudaMemcpyAsync(d_base, chan_base.data(), n_ang * sizeof(long long), cudaMemcpyHostToDevice, s));
  PV(cudaMemcpyAsync(d_nch, nch.data(), n_ang * sizeof(int), cudaMemcpyHostToDevice, s));
  PV(cudaMemcpyAsync(d_pref, rad_pref.data(), (n_rad + 1) * sizeof(int), cudaMemcpyHostToDevice, s));
  p.chan_base = d_base; p.nch = d_nch; p.rad_pref = d_pref;
  const int blocks = tdde_num_sms() * 8;
  k_pv_rowptr<<<blocks, 256, 0, s>>>(p, n, nnz);
  k_pv_assemble<0><<<blocks, 256, 0, s>>>(p, n);                      // structure: once
  h->launches += 2;
  ScopedEvent e0, e1, e2;
  PV(e0.create()); PV(e1.create()); PV(e2.create());
  k_pv_assemble<1><<<blocks, 256, 0, s>>>(p, n);                      // warm-up
  k_pv_spmv<<<blocks, 256, 0, s>>>(p, n, reinterpret_cast<const cplx*>(x_dev), reinterpret_cast<cplx*>(y_dev));
  PV(cudaEventRecord(e0, s));
  for (int r = 0; r < reps; ++r) k_pv_assemble<1><<<blocks, 256, 0, s>>>(p, n);
  PV(cudaEventRecord(e1, s));
  for (int r = 0; r < reps; ++r) k_pv_spmv<<<blocks, 256, 0, s>>>(p, n, reinterpret_cast<const cplx*>(x_dev), reinterpret_cast<cplx*>(y_dev));
  PV(cudaEventRecord(e2, s));
  PV(cudaEventSynchronize(e2));
  h->launches += 2 + 2 * reps;
  float ta = 0, ts = 0;
  PV(cudaEventElapsedTime(&ta, e0, e1));
  PV(cudaEventElapsedTime(&ts, e1, e2));
  if (ms_assemble) *ms_assemble = ta / reps;
  if (ms_spmv) *ms_spmv = ts / reps;
  PV(cudaGetLastError());
#undef PV
  cleanup();
  return 0;
}

#endif  // TDDE_WITH_BENCH
