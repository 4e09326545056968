// tdde_reduce.cuh -- deterministic grid reduction + on-device scalar updates.
//
// Every fused kernel ends the same way: per-thread sums -> warp shuffle tree -> per-warp slots in shared
// memory summed in warp order -> one partial per block in global scratch -> the block that draws the last
// ticket sums the partials in block order and updates the BiCGSTAB scalars in SolverState.  The summation
// order depends only on the launch geometry, so results are bitwise reproducible run to run (pin P12).
#pragma once
#include "tdde_internal.h"

__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
// acc += a * b  (4 DFMA)
__device__ __forceinline__ void cfma(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
// acc -= a * b  (4 DFMA; the negations are operand modifiers)
__device__ __forceinline__ void cfms(cplx& acc, cplx a, cplx b) {
  acc.x = fma(-a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(-a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}
// acc += conj(a) * b
__device__ __forceinline__ void cfma_conj(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}
__device__ __forceinline__ cplx cdiv(cplx a, cplx b) {
  // Smith's algorithm: no overflow for well-scaled data, deterministic
  if (fabs(b.x) >= fabs(b.y)) {
    double r = b.y / b.x, d = b.x + b.y * r;
    return make_double2((a.x + a.y * r) / d, (a.y - a.x * r) / d);
  } else {
    double r = b.x / b.y, d = b.x * r + b.y;
    return make_double2((a.x * r + a.y) / d, (a.y * r - a.x) / d);
  }
}
__device__ __forceinline__ bool cbad(cplx a) {
  double m = fmax(fabs(a.x), fabs(a.y));
  return !(isfinite(a.x) && isfinite(a.y)) || m < TDDE_TINY;
}

// per-thread asynchronous 16-byte copies global -> shared (LDGSTS)
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ bool solver_idle(const SolverState* st) {
  // uniform over the grid: all three are only written by finalisers of earlier kernels
  return st->done | st->stalled | (st->status != 0);
}

// The scalar recurrences of BiCGSTAB, executed by one thread of the last block.
__device__ inline void finalize_scalars(SolverState* st, int fin, double d0x, double d0y, double d1) {
  switch (fin) {
    case FIN_NB: st->nb2 = d1; break;
    case FIN_NORM: st->norm_out = d0x; break;
    case FIN_DOTS: st->rho_old = make_double2(d0x, d0y); st->res2 = d1; break;
    case FIN_RES0: st->res2 = d1; break;
    case FIN_R0S:
      d0x = d1;                                  // ||b||^2 from this kernel, ||r0||^2 from the previous one
      d1 = st->res2;
      // fall through
    case FIN_R0: {
      st->nb2 = d0x;                             // ||b||^2 rides in the first slot
      st->done = 0;
      st->res2 = d1;
      st->rho = make_double2(d1, 0.0);           // rhat = r0  =>  <rhat, r0> = ||r0||^2
      st->rho_old = make_double2(1.0, 0.0);
      st->alpha = make_double2(1.0, 0.0);
      st->omega = make_double2(1.0, 0.0);
      st->beta = make_double2(0.0, 0.0);
      st->first = 1;
      st->half_iters = 0;
      st->half_exit = 0;
      if (!isfinite(d1)) { st->status = TDDE_EBREAKDOWN; st->done = 1; }
      else if (!st->force && d1 <= st->rtol2 * st->nb2) st->done = 1;     // zero iterations
      else if (cbad(st->rho)) { st->status = TDDE_EBREAKDOWN; st->done = 1; }
      break;
    }
    case FIN_ALPHA: {
      cplx rv = make_double2(d0x, d0y);
      st->applies += 1; st->preconds += 1;
      if (cbad(rv)) { st->status = TDDE_EBREAKDOWN; st->done = 1; }
      else st->alpha = cdiv(st->rho, rv);
      break;
    }
    case FIN_S: {
      st->res2 = d1;
      st->half_iters += 1;
      if (!isfinite(d1)) { st->status = TDDE_EBREAKDOWN; st->done = 1; }
      else if (!st->force && d1 <= st->rtol2 * st->nb2) { st->half_exit = 1; st->done = 1; }
      break;
    }
    case FIN_OMEGA: {
      cplx ts = make_double2(d0x, -d0y);         // <t,s> = conj(<s,t>)
      st->applies += 1; st->preconds += 1;
      if (!isfinite(d1) || d1 < TDDE_TINY) { st->status = TDDE_EBREAKDOWN; st->done = 1; }
      else st->omega = make_double2(ts.x / d1, ts.y / d1);
      break;
    }
    case FIN_R: {
      cplx rho_new = make_double2(d0x, d0y);
      st->res2 = d1;
      st->half_iters += 1;
      st->first = 0;
      if (!isfinite(d1)) { st->status = TDDE_EBREAKDOWN; st->done = 1; break; }
      if (!st->force && d1 <= st->rtol2 * st->nb2) { st->done = 1; break; }
      if (!st->force && st->half_iters >= st->max_half) { st->status = TDDE_ENOCONV; st->done = 1; break; }
      if (cbad(rho_new) || cbad(st->omega)) { st->status = TDDE_EBREAKDOWN; st->done = 1; break; }
      st->beta = cmul(cdiv(rho_new, st->rho), cdiv(st->alpha, st->omega));   // (rho/rho_old)(alpha/omega)
      st->rho_old = st->rho;
      st->rho = rho_new;
      break;
    }
    default: break;
  }
}

// v[0..2] = (Re d0, Im d0, d1) per thread.  Must be called by every thread of every block of the grid.
// NT = threads per block (multiple of 32, <= 1024).
template <int NT>
__device__ __forceinline__ void grid_reduce_finalize(double v0, double v1, double v2, const ReduceCtx& rc) {
  __shared__ double sm[3][NT / 32];
  __shared__ bool is_last;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    v0 += __shfl_down_sync(0xffffffffu, v0, o);
    v1 += __shfl_down_sync(0xffffffffu, v1, o);
    v2 += __shfl_down_sync(0xffffffffu, v2, o);
  }
  if (lane == 0) { sm[0][wid] = v0; sm[1][wid] = v1; sm[2][wid] = v2; }
  __syncthreads();
  const unsigned nblk = gridDim.x * gridDim.y;
  const unsigned bid = blockIdx.y * gridDim.x + blockIdx.x;
  if (threadIdx.x == 0) {
    double a = 0, b = 0, c = 0;
    for (int k = 0; k < NT / 32; ++k) { a += sm[0][k]; b += sm[1][k]; c += sm[2][k]; }
    double* p = rc.partials + 4 * (size_t)bid;
    p[0] = a; p[1] = b; p[2] = c;
    __threadfence();
    unsigned t = atomicAdd(rc.ticket, 1u);
    is_last = (t == nblk - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double a = 0, b = 0, c = 0;
  for (unsigned k = threadIdx.x; k < nblk; k += NT) {      // fixed order per thread
    const volatile double* p = rc.partials + 4 * (size_t)k;
    a += p[0]; b += p[1]; c += p[2];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_down_sync(0xffffffffu, a, o);
    b += __shfl_down_sync(0xffffffffu, b, o);
    c += __shfl_down_sync(0xffffffffu, c, o);
  }
  __syncthreads();
  if (lane == 0) { sm[0][wid] = a; sm[1][wid] = b; sm[2][wid] = c; }
  __syncthreads();
  if (threadIdx.x == 0) {
    a = b = c = 0;
    for (int k = 0; k < NT / 32; ++k) { a += sm[0][k]; b += sm[1][k]; c += sm[2][k]; }
    if (rc.shard_out) { rc.shard_out[0] = a; rc.shard_out[1] = b; rc.shard_out[2] = c; }
    else finalize_scalars(rc.st, rc.fin, a, b, c);
    *rc.ticket = 0u;
    __threadfence();
  }
}
