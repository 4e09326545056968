// tdde_vec.cu -- fused BiCGSTAB vector kernels (a3 is fused into the start-of-step applies), layout transposes, small helpers.
//
// All of these are HBM-bound streaming kernels: 128-bit (double2) coalesced loads/stores, grid-stride over
// the internal element count, grid = a fixed multiple of the SM count, the inner products fused into the pass
// that produces the vector and finished by the deterministic grid reduction of tdde_reduce.cuh.
#include "tdde_reduce.cuh"

#define VEC_NT 256
#define VEC_BLOCKS_PER_SM 8
// multiprocessor count of the current device (cached per device)
int tdde_num_sms() {
  static int cache[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
  if (cache[dev] == 0) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    cache[dev] = n;
  }
  return cache[dev];
}
#define NUM_SMS tdde_num_sms()

static int vec_grid(long long n) {
  long long need = (n + VEC_NT - 1) / VEC_NT;
  long long cap = (long long)NUM_SMS * VEC_BLOCKS_PER_SM;
  return (int)(need < cap ? (need < 1 ? 1 : need) : cap);
}

__device__ __forceinline__ cplx ldcs(const cplx* p) { return __ldcs(p); }

// p = r + beta (p - omega v);  first iteration: p = r                                         (a6 i)
__global__ void __launch_bounds__(VEC_NT) k_vec_p(VecArgs a) {
  const SolverState* st = a.red.st;
  if (solver_idle(st)) return;
  const bool first = st->first;
  const cplx beta = st->beta, omega = st->omega;
  for (long long i = (long long)blockIdx.x * VEC_NT + threadIdx.x; i < a.n; i += (long long)gridDim.x * VEC_NT) {
    cplx r = a.r[i];
    if (first) { a.p[i] = r; continue; }
    cplx p = a.p[i], v = a.v[i];
    cplx q = p;                       // q = p - omega v
    cfma(q, make_double2(-omega.x, -omega.y), v);
    cfma(r, beta, q);
    a.p[i] = r;
  }
}

// s = r - alpha v, ||s||^2                                                                   (a6 ii)
__global__ void __launch_bounds__(VEC_NT) k_vec_s(VecArgs a) {
  const SolverState* st = a.red.st;
  if (solver_idle(st)) return;
  const cplx nalpha = make_double2(-st->alpha.x, -st->alpha.y);
  double s2 = 0;
  for (long long i = (long long)blockIdx.x * VEC_NT + threadIdx.x; i < a.n; i += (long long)gridDim.x * VEC_NT) {
    cplx s = a.r[i], v = a.v[i];
    cfma(s, nalpha, v);
    a.s[i] = s;
    s2 = fma(s.x, s.x, s2); s2 = fma(s.y, s.y, s2);
  }
  grid_reduce_finalize<VEC_NT>(0.0, 0.0, s2, a.red);
}

// half-step exit: x += alpha y, only when FIN_S latched half_exit == 1                        (C4, C8-11)
__global__ void __launch_bounds__(VEC_NT) k_vec_halfexit(VecArgs a) {
  SolverState* st = a.red.st;
  if (st->half_exit != 1 || st->stalled || st->status != 0) return;
  const cplx alpha = st->alpha;
  for (long long i = (long long)blockIdx.x * VEC_NT + threadIdx.x; i < a.n; i += (long long)gridDim.x * VEC_NT) {
    cplx x = a.x[i];
    cfma(x, alpha, a.y[i]);
    a.x[i] = x;
  }
  __shared__ bool last;
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    last = (atomicAdd(a.red.ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (last && threadIdx.x == 0) { st->half_exit = 2; *a.red.ticket = 0u; __threadfence(); }
}

// x += alpha y + omega z;  r = s - omega t;  <rhat, r>, ||r||^2                               (a6 iii)
__global__ void __launch_bounds__(VEC_NT) k_vec_xr(VecArgs a) {
  const SolverState* st = a.red.st;
  if (solver_idle(st)) return;
  const cplx alpha = st->alpha, omega = st->omega;
  const cplx nomega = make_double2(-omega.x, -omega.y);
  cplx d0 = make_double2(0, 0);
  double r2 = 0;
  for (long long i = (long long)blockIdx.x * VEC_NT + threadIdx.x; i < a.n; i += (long long)gridDim.x * VEC_NT) {
    cplx x = a.x[i];
    cfma(x, alpha, a.y[i]);
    cfma(x, omega, a.z[i]);
    a.x[i] = x;
    cplx r = a.s[i];
    cfma(r, nomega, a.t[i]);
    a.r[i] = r;
    cfma_conj(d0, a.rhat[i], r);
    r2 = fma(r.x, r.x, r2); r2 = fma(r.y, r.y, r2);
  }
  grid_reduce_finalize<VEC_NT>(d0.x, d0.y, r2, a.red);
}

__global__ void k_step_open(SolverState* st, int step_idx, int force, int clear_stall_only) {
  if (clear_stall_only) { st->stalled = 0; return; }
  st->step_idx = step_idx; st->force = force; st->done = 0; st->stalled = 0; st->half_exit = 0;
  st->steps_done = 0; st->total_half = 0; st->applies = 0; st->preconds = 0;
  st->last_half_iters = 0; st->last_rel_res = 0.0;
}

__global__ void k_step_close(SolverState* st) {
  if (st->stalled || st->status != 0) return;
  if (!st->done) { st->stalled = 1; return; }
  st->steps_done += 1;
  st->total_half += st->half_iters;
  st->last_half_iters = st->half_iters;
  st->last_rel_res = st->nb2 > 0 ? sqrt(st->res2 / st->nb2) : 0.0;
  st->step_idx += 1;
  st->applies += 2;              // the two start-of-step applies (H c and S c)
}

// ---- layout transposes: boundary c[a * n_rad + j]  <->  internal X[j * ld + a] (pads zeroed) ----
#define TP 32
__global__ void __launch_bounds__(TP * 8) k_to_internal(const cplx* __restrict__ c, cplx* __restrict__ X,
                                                         int n_ang, int n_rad, int ld) {
  __shared__ cplx tile[TP][TP + 1];
  const int a0 = blockIdx.x * TP, j0 = blockIdx.y * TP;
  for (int r = threadIdx.y; r < TP; r += 8) {          // read: rows = channels, fast = radial
    int a = a0 + r, j = j0 + threadIdx.x;
    tile[r][threadIdx.x] = (a < n_ang && j < n_rad) ? c[(size_t)a * n_rad + j] : make_double2(0, 0);
  }
  __syncthreads();
  for (int r = threadIdx.y; r < TP; r += 8) {          // write: rows = radial, fast = channels
    int j = j0 + r, a = a0 + threadIdx.x;
    if (j < n_rad && a < ld) X[(size_t)j * ld + a] = tile[threadIdx.x][r];
  }
}
__global__ void __launch_bounds__(TP * 8) k_to_boundary(const cplx* __restrict__ X, cplx* __restrict__ c,
                                                         int n_ang, int n_rad, int ld) {
  __shared__ cplx tile[TP][TP + 1];
  const int a0 = blockIdx.x * TP, j0 = blockIdx.y * TP;
  for (int r = threadIdx.y; r < TP; r += 8) {
    int j = j0 + r, a = a0 + threadIdx.x;
    tile[r][threadIdx.x] = (j < n_rad && a < n_ang) ? X[(size_t)j * ld + a] : make_double2(0, 0);
  }
  __syncthreads();
  for (int r = threadIdx.y; r < TP; r += 8) {
    int a = a0 + r, j = j0 + threadIdx.x;
    if (a < n_ang && j < n_rad) c[(size_t)a * n_rad + j] = tile[threadIdx.x][r];
  }
}

__global__ void k_combine(const cplx* __restrict__ S, const cplx* __restrict__ H0, cplx alpha, cplx beta,
                          cplx* __restrict__ out, long long count) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x) {
    cplx o = cmul(alpha, S[i]);
    cfma(o, beta, H0[i]);
    out[i] = o;
  }
}

__global__ void k_fill(cplx* v, long long n, unsigned seed) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    unsigned h = (unsigned)(i * 2654435761u) ^ seed; h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
    unsigned q = h * 3266489917u; q ^= q >> 16;
    v[i] = make_double2((h & 0xffff) / 32768.0 - 1.0, (q & 0xffff) / 32768.0 - 1.0);
  }
}
int launch_fill(cplx* v, long long n, unsigned seed, cudaStream_t s) { k_fill<<<NUM_SMS * 8, 256, 0, s>>>(v, n, seed); return 1; }

// FP64 FMA peak probe: 8 independent chains per thread, all SMs
__global__ void __launch_bounds__(256) k_dfma_peak(double* out, int iters) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999, c = 1e-7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) out[0] = s;
}

// FP64 pipe probe (DESIGN.md 4.1 (1b)): mode 1 = DMMA only (mma.sync.m8n8k4.f64, 8 independent accumulators), mode 2 = per iteration
// 8 DMMAs followed by 32 DFMAs in the same warp -- the mix of k_apply_mma.  One flop count for both: 2 x 256 per DMMA, 2 x 32 per DFMA.
__global__ void __launch_bounds__(256) k_fp64_pipe_probe(double* out, int iters, int mode) {
  double c[8][2], f[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { c[i][0] = 0; c[i][1] = 0; f[i] = i; }
  const double a = threadIdx.x * 1e-3, b = threadIdx.x * 2e-3, m = 0.999999, k = 1e-7;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    if (mode == 2) {
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(f[i]) : "d"(m), "d"(k));
    }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1] + f[i];
  if (s == 123.456) out[0] = s;
}
int launch_fp64_pipe_probe(double* out, int blocks, int threads, int iters, int mode, cudaStream_t s) {
  k_fp64_pipe_probe<<<blocks, threads, 0, s>>>(out, iters, mode); return 1;
}

int launch_vec_p(const VecArgs& a, cudaStream_t s) { k_vec_p<<<vec_grid(a.n), VEC_NT, 0, s>>>(a); return 1; }
int launch_vec_s(const VecArgs& a, cudaStream_t s) { k_vec_s<<<vec_grid(a.n), VEC_NT, 0, s>>>(a); return 1; }
int launch_vec_halfexit(const VecArgs& a, cudaStream_t s) { k_vec_halfexit<<<vec_grid(a.n), VEC_NT, 0, s>>>(a); return 1; }
int launch_vec_xr(const VecArgs& a, cudaStream_t s) { k_vec_xr<<<vec_grid(a.n), VEC_NT, 0, s>>>(a); return 1; }
int launch_step_open(SolverState* st, int step_idx, int force, int clear_stall_only, cudaStream_t s) {
  k_step_open<<<1, 1, 0, s>>>(st, step_idx, force, clear_stall_only); return 1;
}
int launch_step_close(SolverState* st, cudaStream_t s) { k_step_close<<<1, 1, 0, s>>>(st); return 1; }
int launch_to_internal(const cplx* c, cplx* X, int n_ang, int n_rad, int ld, cudaStream_t s) {
  dim3 g((ld + TP - 1) / TP, (n_rad + TP - 1) / TP), b(TP, 8);
  k_to_internal<<<g, b, 0, s>>>(c, X, n_ang, n_rad, ld); return 1;
}
int launch_to_boundary(const cplx* X, cplx* c, int n_ang, int n_rad, int ld, cudaStream_t s) {
  dim3 g((ld + TP - 1) / TP, (n_rad + TP - 1) / TP), b(TP, 8);
  k_to_boundary<<<g, b, 0, s>>>(X, c, n_ang, n_rad, ld); return 1;
}
int launch_combine_blocks(const cplx* S, const cplx* H0, cplx alpha, cplx beta, cplx* out, long long count, cudaStream_t s) {
  long long nb = (count + 255) / 256; if (nb > NUM_SMS * 8) nb = NUM_SMS * 8; if (nb < 1) nb = 1;
  k_combine<<<(int)nb, 256, 0, s>>>(S, H0, alpha, beta, out, count); return 1;
}
int launch_dfma_peak(double* out, int blocks, int threads, int iters, cudaStream_t s) {
  k_dfma_peak<<<blocks, threads, 0, s>>>(out, iters); return 1;
}
