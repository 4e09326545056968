// tdde_noalloc.cu -- tdde_snorm_noalloc: Re(c^H S c) (tdde_norm's quantity; S: PAPER.md:178-182) for callers that cannot allocate:
// no handle, no cudaMalloc / cudaFree, no allocating library call (include/tdde.h states the contract).
//
// It is the S-only apply with its fused norm reduction.  The handle path (k_apply_banded<0, ...> + grid_reduce_finalize) keeps the
// per-block partial sums and the completion ticket of that reduction in buffers allocated by tdde_create; here they live in the
// file-scope array below, a fixed 64 KB + 256 B of device memory per GPU that loads the library.  In host code the array's NAME is only
// a host-side stand-in for the symbol, not a device address: the address is resolved once per device with cudaGetSymbolAddress (with that
// device current) and it is that pointer the kernel gets.
// Every call on a device shares the array and finds the previous call's contents in it: the ticket is cleared by a memset node at the
// start of each call (and again by the finishing block), every partial that is read has been written by the same launch.  Calls that
// overlap on the GPU race on it.
#include <string>
#include "tdde_handle.h"
#include "tdde_reduce.cuh"

#define NA_NT 256
#define NA_EPT (TDDE_NOALLOC_ELEMS_PER_BLOCK / NA_NT)
#define NA_MAXW 32

// [0, MAX_BLOCKS): one partial sum per block; [MAX_BLOCKS]: the completion ticket (an unsigned int in the first 4 bytes)
static __device__ __align__(256) double g_noalloc_scratch[TDDE_NOALLOC_MAX_BLOCKS + 32];

// fixed-order block sum of one double per thread; result valid in thread 0
__device__ __forceinline__ double na_block_sum(double v, double* sm) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  __syncthreads();                                     // sm may still be read from an earlier use
  if (lane == 0) sm[wid] = v;
  __syncthreads();
  double s = 0;
  if (threadIdx.x == 0)
    for (int k = 0; k < NA_NT / 32; ++k) s += sm[k];
  return s;
}

// One thread per element e = a * n_rad + i (boundary layout: consecutive threads walk the radial index, coalesced):
//   u = sum_d S_{k(a)}[i][i + d] c[a][i + d],  acc += Re(conj(c[a][i]) u).
// Block b owns elements [b, b + 1) * ELEMS_PER_BLOCK; its sum goes to scratch[b]; the block that draws the last ticket adds the
// partials in block order (deterministic) and writes *out.
__global__ void __launch_bounds__(NA_NT) k_snorm_noalloc(int n_ang, int n_rad, int w0, const cplx* __restrict__ S, const int* __restrict__ cls,
                                                         const cplx* __restrict__ c, double* __restrict__ out, double* scratch) {
  __shared__ double sm[NA_NT / 32];
  __shared__ bool is_last;
  const long long n = (long long)n_ang * n_rad;
  const long long base = (long long)blockIdx.x * TDDE_NOALLOC_ELEMS_PER_BLOCK;
  const int nd = 2 * w0 + 1;
  double acc = 0;
#pragma unroll
  for (int q = 0; q < NA_EPT; ++q) {
    const long long e = base + (long long)q * NA_NT + threadIdx.x;
    if (e < n) {
      const int a = (int)(e / n_rad), i = (int)(e % n_rad);
      const cplx* row = S + ((size_t)cls[a] * n_rad + i) * nd + w0;
      const cplx* ca = c + (size_t)a * n_rad;
      cplx u = make_double2(0, 0);
      const int dlo = max(-w0, -i), dhi = min(w0, n_rad - 1 - i);
      for (int d = dlo; d <= dhi; ++d) cfma(u, row[d], ca[i + d]);
      const cplx ci = ca[i];
      acc = fma(ci.x, u.x, acc);
      acc = fma(ci.y, u.y, acc);
    }
  }
  const double bsum = na_block_sum(acc, sm);
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + TDDE_NOALLOC_MAX_BLOCKS);
  if (threadIdx.x == 0) {
    scratch[blockIdx.x] = bsum;
    __threadfence();
    is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double t = 0;
  for (unsigned k = threadIdx.x; k < gridDim.x; k += NA_NT) t += reinterpret_cast<const volatile double*>(scratch)[k];   // fixed order per thread
  const double tot = na_block_sum(t, sm);
  if (threadIdx.x == 0) {
    out[0] = tot;
    *ticket = 0u;                                      // leave the array ready for the next call
  }
}

// ---- host side ----
static double* g_noalloc_ptr[64] = {};                 // device address of g_noalloc_scratch, per device

static int noalloc_resolve(double** ptr) {
  int dev = -1;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) { g_last_cuda_error = "tdde_snorm_noalloc: device ordinal outside [0, 64)"; return TDDE_EINVAL; }
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);      // the symbol's address on the CURRENT device
    if (e != cudaSuccess) return tdde_cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
    if (!p) { g_last_cuda_error = "cudaGetSymbolAddress(g_noalloc_scratch) returned a null address"; return TDDE_ECUDA; }
    g_noalloc_ptr[dev] = static_cast<double*>(p);
  }
  *ptr = g_noalloc_ptr[dev];
  return 0;
}

extern "C" int tdde_snorm_noalloc_setup(void) {
  double* p = nullptr;
  return noalloc_resolve(&p);
}

extern "C" int tdde_snorm_noalloc(int32_t n_ang, int32_t n_rad, int32_t n_cls, int32_t w0, const tdde_c64* S_band_dev, const int32_t* cls_dev,
                                  const tdde_c64* c_dev, double* out_dev, void* cuda_stream) {
  if (n_ang <= 0 || n_rad <= 0 || n_cls <= 0 || w0 < 0 || w0 > NA_MAXW || w0 >= n_rad || !S_band_dev || !cls_dev || !c_dev || !out_dev) {
    g_last_cuda_error = "tdde_snorm_noalloc: null pointer, non-positive dimension, or w0 outside [0, min(32, n_rad - 1)]";
    return TDDE_EINVAL;
  }
  const long long n = (long long)n_ang * n_rad;
  if (n > (long long)TDDE_NOALLOC_MAX_N) {
    g_last_cuda_error = "tdde_snorm_noalloc: n_ang * n_rad = " + std::to_string(n) + " exceeds TDDE_NOALLOC_MAX_N = " +
                        std::to_string((long long)TDDE_NOALLOC_MAX_N) + " (the static scratch array holds one partial sum per " +
                        std::to_string(TDDE_NOALLOC_ELEMS_PER_BLOCK) + " elements, " + std::to_string(TDDE_NOALLOC_MAX_BLOCKS) + " at most)";
    return TDDE_EINVAL;
  }
  double* scratch = nullptr;
  int rc = noalloc_resolve(&scratch);
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int nblk = (int)((n + TDDE_NOALLOC_ELEMS_PER_BLOCK - 1) / TDDE_NOALLOC_ELEMS_PER_BLOCK);
  // the ticket must start at zero whatever an earlier (possibly aborted) call left behind; partials need no clearing: block b of this
  // launch writes scratch[b] before the finishing block reads it
  CU(cudaMemsetAsync(scratch + TDDE_NOALLOC_MAX_BLOCKS, 0, 256, s));
  k_snorm_noalloc<<<nblk, NA_NT, 0, s>>>(n_ang, n_rad, w0, reinterpret_cast<const cplx*>(S_band_dev), cls_dev, reinterpret_cast<const cplx*>(c_dev),
                                         out_dev, scratch);
  CU(cudaGetLastError());
  return 0;
}
