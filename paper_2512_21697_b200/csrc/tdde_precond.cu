// tdde_precond.cu -- y = (S + i dt/2 H0)^{-1} x as batched banded triangular solves (
// PAPER.md:211-215, Eq. 26: M is block-diagonal over angular channels, LU factors computed at start-up).
//
// One thread per angular channel, lanes = consecutive channels (coalesced 16-byte accesses in the internal
// layout).  Both sweeps run in column-oriented (axpy) form: once y_i is final, the W pending rows below it
// are updated independently, so the dependent chain per row is a single complex FMA and the remaining W-1
// updates are instruction-level parallel.  Unit-lower L: Lcol[k][i][d-1] = L[i+d][i];  U: Ucol[k][i][0] =
// 1/U[i][i], Ucol[k][i][d] = U[i-d][i].  Coefficients are per-lane loads indexed by the channel's class;
// lanes of the same class hit the same address.  Loads for row block n+1 are issued before the dependent
// chain of block n (software prefetch), because the recurrence itself cannot be parallelised along r.
#include "tdde_reduce.cuh"

#define PC_NT 32
#define PC_UNROLL 4

template <int W>
__global__ void __launch_bounds__(PC_NT) k_precond(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * PC_NT + threadIdx.x;
  if (a >= p.ld) return;
  const int ld = p.ld, n_rad = p.n_rad;
  const int k = p.cls[a];
  const cplx* Lc = p.Lcol + (size_t)k * n_rad * W;
  const cplx* Uc = p.Ucol + (size_t)k * n_rad * (W + 1);

  cplx pw[W + 1];
#pragma unroll
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);

  // ---- forward: L y = x ----
  {
    cplx xn[PC_UNROLL], cn[PC_UNROLL][W];
    auto load = [&](int ib) {
#pragma unroll
      for (int u = 0; u < PC_UNROLL; ++u) {
        const int i = min(ib + u, n_rad - 1);
        xn[u] = p.x[(size_t)i * ld + a];
#pragma unroll
        for (int d = 0; d < W; ++d) cn[u][d] = __ldg(Lc + (size_t)i * W + d);
      }
    };
    load(0);
    for (int ib = 0; ib < n_rad; ib += PC_UNROLL) {
      cplx xc[PC_UNROLL], cc[PC_UNROLL][W];
#pragma unroll
      for (int u = 0; u < PC_UNROLL; ++u) {
        xc[u] = xn[u];
#pragma unroll
        for (int d = 0; d < W; ++d) cc[u][d] = cn[u][d];
      }
      if (ib + PC_UNROLL < n_rad) load(ib + PC_UNROLL);
#pragma unroll
      for (int u = 0; u < PC_UNROLL; ++u) {
        const int i = ib + u;
        if (i < n_rad) {
          const cplx yi = cadd(xc[u], pw[0]);
          p.y[(size_t)i * ld + a] = yi;
          const cplx nyi = make_double2(-yi.x, -yi.y);
#pragma unroll
          for (int d = 0; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], cc[u][d], nyi); }
        }
      }
    }
  }
#pragma unroll
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
  // ---- backward: U x = y ----
  {
    cplx xn[PC_UNROLL], cn[PC_UNROLL][W + 1];
    auto load = [&](int ib) {          // rows ib, ib-1, ...
#pragma unroll
      for (int u = 0; u < PC_UNROLL; ++u) {
        const int i = max(ib - u, 0);
        xn[u] = p.y[(size_t)i * ld + a];
#pragma unroll
        for (int d = 0; d <= W; ++d) cn[u][d] = __ldg(Uc + (size_t)i * (W + 1) + d);
      }
    };
    load(n_rad - 1);
    for (int ib = n_rad - 1; ib >= 0; ib -= PC_UNROLL) {
      cplx xc[PC_UNROLL], cc[PC_UNROLL][W + 1];
#pragma unroll
      for (int u = 0; u < PC_UNROLL; ++u) {
        xc[u] = xn[u];
#pragma unroll
        for (int d = 0; d <= W; ++d) cc[u][d] = cn[u][d];
      }
      if (ib - PC_UNROLL >= 0) load(ib - PC_UNROLL);
#pragma unroll
      for (int u = 0; u < PC_UNROLL; ++u) {
        const int i = ib - u;
        if (i >= 0) {
          const cplx xi = cmul(cadd(xc[u], pw[0]), cc[u][0]);
          p.y[(size_t)i * ld + a] = xi;
          const cplx nxi = make_double2(-xi.x, -xi.y);
#pragma unroll
          for (int d = 0; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], cc[u][d + 1], nxi); }
        }
      }
    }
  }
}

// runtime-w fallback (w <= 32): pending rows in a small circular local array
__global__ void __launch_bounds__(PC_NT) k_precond_any(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * PC_NT + threadIdx.x;
  if (a >= p.ld) return;
  const int ld = p.ld, n_rad = p.n_rad, W = p.w;
  const int k = p.cls[a];
  const cplx* Lc = p.Lcol + (size_t)k * n_rad * W;
  const cplx* Uc = p.Ucol + (size_t)k * n_rad * (W + 1);
  cplx pw[33];
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
  for (int i = 0; i < n_rad; ++i) {
    const cplx yi = cadd(p.x[(size_t)i * ld + a], pw[0]);
    p.y[(size_t)i * ld + a] = yi;
    const cplx nyi = make_double2(-yi.x, -yi.y);
    for (int d = 0; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], Lc[(size_t)i * W + d], nyi); }
  }
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
  for (int i = n_rad - 1; i >= 0; --i) {
    const cplx* uc = Uc + (size_t)i * (W + 1);
    const cplx xi = cmul(cadd(p.y[(size_t)i * ld + a], pw[0]), uc[0]);
    p.y[(size_t)i * ld + a] = xi;
    const cplx nxi = make_double2(-xi.x, -xi.y);
    for (int d = 0; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], uc[d + 1], nxi); }
  }
}

int launch_precond(const PrecArgs& a, cudaStream_t s) {
  const int grid = (a.ld + PC_NT - 1) / PC_NT;
  switch (a.w) {
    case 3: k_precond<3><<<grid, PC_NT, 0, s>>>(a); break;
    case 6: k_precond<6><<<grid, PC_NT, 0, s>>>(a); break;
    case 9: k_precond<9><<<grid, PC_NT, 0, s>>>(a); break;
    case 13: k_precond<13><<<grid, PC_NT, 0, s>>>(a); break;
    default:
      if (a.w > 32 || a.w < 1) return -1;
      k_precond_any<<<grid, PC_NT, 0, s>>>(a);
  }
  return 1;
}
