// tdde_precond.cu -- y = (S + i dt/2 H0)^{-1} x as batched banded solves (
// PAPER.md:211-215, Eq. 26: M is block-diagonal over angular channels, LU factors computed at start-up).
//
// The radial index is cut into P interiors separated by P-1 separators of w rows (tdde_partition.h); the solve is an
// exact reordering of Gaussian elimination in three kernels:
//   P1  k_precond_spikes   r(-)_q, r(+)_q = W b_I : streaming, 2 w complex FMAs per interior row, one read of b
//   P2  k_precond_schur    block-Thomas solve of the block-tridiagonal Schur system for the separator unknowns
//   P3  k_precond_tile     per (32 channels x interior): b_I - A_IS x_S into a SHARED-MEMORY tile, L sweep and U sweep on
//                          the tile, one coalesced write of x_I.  No intermediate vector ever goes to global memory.
// Algorithmic traffic: 16 B (P1) + 32 B (P3) per element instead of 96 B for sweep / store / reload / correct.
// One warp per 32 consecutive channels, lane = channel (coalesced 16-byte accesses in the internal layout).  Both
// sweeps run in column-oriented (axpy) form: once y_i is final the W pending rows below it are updated independently;
// only the update of the next row is on the critical path, and it is split as  pw0' = (pw1 - c x_i) - c pw0  so that
// the chain is one complex FMA (two dependent DFMAs) per row; for the U sweep the host pre-scales U[i-1][i] by
// 1/U[i][i] for the same reason.  Factor rows of the (few) kappa-classes present in the warp stream through a
// cp.async ring in shared memory.
// Factor layout (tdde_partition.cu): Lcol[k][i][d-1] = L[i+d][i];
//   Ucol[k][i][0] = 1/U[i][i], Ucol[k][i][1] = U[i-1][i] / U[i][i], Ucol[k][i][d>=2] = U[i-d][i].
#include "tdde_reduce.cuh"

#define PC_NT 32
#define PC_ROWS 8
#define PC_STAGES 2
#define PC_MAXC TDDE_PC_MAXC

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int W>
struct PrecPlan {
  static constexpr int CW = W + 1;                                   // coefficient row width (U needs W+1)
  static constexpr int STAGE = PC_MAXC * PC_ROWS * CW;               // complex per stage (factor rows only)
  static constexpr int RING = PC_STAGES * STAGE;                     // complex
  static size_t smem(int tile_rows) { return ((size_t)RING + (size_t)tile_rows * PC_NT) * sizeof(cplx); }
};

// ---- P1: spike dot products.  CTA = 128 channels x one interior; thread = channel. ----
template <int W>
__global__ void __launch_bounds__(128) k_precond_spikes(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * 128 + threadIdx.x;
  if (a >= p.ld) return;
  const int q = blockIdx.y, ld = p.ld;
  const int lo = p.plo[q], hi = p.phi[q];
  const bool has_m = q > 0, has_p = q + 1 < p.P;
  const cplx* Wk = p.Wsp + (size_t)p.cls[a] * p.n_rad * 2 * W;
  const cplx* xin = p.x + a;
  cplx am[W], ap[W];
#pragma unroll
  for (int c = 0; c < W; ++c) am[c] = ap[c] = make_double2(0, 0);
  int i = lo;
  for (; i + 4 <= hi; i += 4) {
    cplx b[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) b[u] = xin[(size_t)(i + u) * ld];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const cplx* wr = Wk + (size_t)(i + u) * 2 * W;
      if (has_m) {
#pragma unroll
        for (int c = 0; c < W; ++c) cfma(am[c], __ldg(wr + c), b[u]);
      }
      if (has_p) {
#pragma unroll
        for (int c = 0; c < W; ++c) cfma(ap[c], __ldg(wr + W + c), b[u]);
      }
    }
  }
  for (; i < hi; ++i) {
    const cplx b = xin[(size_t)i * ld];
    const cplx* wr = Wk + (size_t)i * 2 * W;
#pragma unroll
    for (int c = 0; c < W; ++c) { cfma(am[c], __ldg(wr + c), b); cfma(ap[c], __ldg(wr + W + c), b); }
  }
#pragma unroll
  for (int c = 0; c < W; ++c) {
    p.rsm[((size_t)q * W + c) * ld + a] = am[c];
    p.rsp[((size_t)q * W + c) * ld + a] = ap[c];
  }
}

// ---- P2: block Thomas over the separators; thread = channel.  r_j = b_S(j) - r(+)_j - r(-)_{j+1};
// forward r'_j = r_j - (B_j D'^-1_{j-1}) r'_{j-1} (kept in the r(+) scratch), backward x_j = D'^-1_j (r'_j - C_j x_{j+1}). ----
template <int W>
__global__ void __launch_bounds__(PC_NT) k_precond_schur(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * PC_NT + threadIdx.x;
  const int ld = p.ld, ns = p.P - 1;
  constexpr int WW = W * W;
  const cplx* Sk = p.Schur + (size_t)p.cls[a] * ns * 3 * WW;
  cplx prev[W], r[W];
#pragma unroll
  for (int c = 0; c < W; ++c) prev[c] = make_double2(0, 0);
  for (int j = 0; j < ns; ++j) {
    const int s0 = p.phi[j];
#pragma unroll
    for (int c = 0; c < W; ++c) {
      const cplx b = p.x[(size_t)(s0 + c) * ld + a];
      const cplx m1 = p.rsp[((size_t)j * W + c) * ld + a], m2 = p.rsm[((size_t)(j + 1) * W + c) * ld + a];
      r[c] = make_double2(b.x - m1.x - m2.x, b.y - m1.y - m2.y);
    }
    if (j > 0) {
      const cplx* Lb = Sk + (size_t)j * 3 * WW;
#pragma unroll
      for (int c = 0; c < W; ++c)
#pragma unroll
        for (int k = 0; k < W; ++k) {
          const cplx l = __ldg(Lb + c * W + k);
          cfma(r[c], make_double2(-l.x, -l.y), prev[k]);
        }
    }
#pragma unroll
    for (int c = 0; c < W; ++c) { p.rsp[((size_t)j * W + c) * ld + a] = r[c]; prev[c] = r[c]; }
  }
  cplx xn[W];
#pragma unroll
  for (int c = 0; c < W; ++c) xn[c] = make_double2(0, 0);
  for (int j = ns - 1; j >= 0; --j) {
    const cplx* Di = Sk + (size_t)j * 3 * WW + WW;
    const cplx* Cj = Di + WW;
#pragma unroll
    for (int c = 0; c < W; ++c) r[c] = p.rsp[((size_t)j * W + c) * ld + a];
    if (j + 1 < ns) {
#pragma unroll
      for (int c = 0; c < W; ++c)
#pragma unroll
        for (int k = 0; k < W; ++k) {
          const cplx l = __ldg(Cj + c * W + k);
          cfma(r[c], make_double2(-l.x, -l.y), xn[k]);
        }
    }
    const int s0 = p.phi[j];
#pragma unroll
    for (int c = 0; c < W; ++c) {
      cplx xv = make_double2(0, 0);
#pragma unroll
      for (int k = 0; k < W; ++k) cfma(xv, __ldg(Di + c * W + k), r[k]);
      prev[c] = xv;
    }
#pragma unroll
    for (int c = 0; c < W; ++c) { xn[c] = prev[c]; p.y[(size_t)(s0 + c) * ld + a] = prev[c]; }
  }
}

// ---- P3: one warp = 32 channels x one interior.  The right-hand side lives in a shared-memory tile (one column per lane, so
// no inter-lane hazards) from its load to the end of the U sweep; factor rows of the warp's kappa-classes stream through a
// cp.async ring. ----
template <int W>
__global__ void __launch_bounds__(PC_NT) k_precond_tile(const PrecArgs p) {
  using PL = PrecPlan<W>;
  if (p.st && solver_idle(p.st)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* ring = reinterpret_cast<cplx*>(smem_raw);
  const int lane = threadIdx.x;
  cplx* tile = ring + PL::RING + lane;                               // this lane's column: tile[r * 32]
  const int a = blockIdx.x * PC_NT + lane;                           // a < ld always (ld is a multiple of 32)
  const int ld = p.ld, n_tot = p.n_rad, q = blockIdx.y;
  const int row0 = p.plo[q];
  const int n_rad = p.phi[q] - row0;                                 // rows of this interior
  const cplx* xin = p.x + (size_t)row0 * ld + a;
  cplx* yout = p.y + (size_t)row0 * ld + a;
  const int* wcls = p.warp_cls + blockIdx.x * PC_MAXC;
  int ncls = 0;
#pragma unroll
  for (int c = 0; c < PC_MAXC; ++c) ncls += (wcls[c] >= 0);
  const int slot = p.slot[a];
  const int k = p.cls[a];
  const int nst = (n_rad + PC_ROWS - 1) / PC_ROWS;

  // right-hand side rows -> tile (asynchronous, all rows in flight at once)
  for (int r = 0; r < n_rad; ++r) cp_async16(tile + r * PC_NT, xin + (size_t)r * ld);
  cp_async_commit();

  cplx pw[W + 1];

  // ================= forward: L y = b_I - A_IS x_S =================
  {
    auto issue = [&](int s) {                                        // factor rows [s*R, s*R + R) of every class
      if (s < nst) {
        cplx* st = ring + (size_t)(s % PC_STAGES) * PL::STAGE;
        const int r0 = s * PC_ROWS, nr = min(PC_ROWS, n_rad - r0);
        for (int c = 0; c < ncls; ++c) {
          const cplx* src = p.Lcol + ((size_t)wcls[c] * n_tot + row0 + r0) * W;
          cplx* dst = st + (size_t)c * PC_ROWS * PL::CW;
          for (int e = lane; e < nr * W; e += PC_NT) cp_async16(dst + e, src + e);
        }
      }
      cp_async_commit();
    };
    for (int s = 0; s < PC_STAGES - 1; ++s) issue(s);
    // separator solutions next to this interior and the corner blocks of A_IS (tdde_partition.h)
    if (p.P > 1) {
      constexpr int WW = W * W;
      const cplx* Ck = p.Corner + ((size_t)k * p.P + q) * 2 * WW;
      cplx xs[W];
      cp_async_wait<PC_STAGES - 1>();                                // the tile has landed (own column: no warp sync needed)
      if (q > 0) {
        const cplx* ys = p.y + (size_t)p.phi[q - 1] * ld + a;
#pragma unroll
        for (int c = 0; c < W; ++c) { const cplx v = ys[(size_t)c * ld]; xs[c] = make_double2(-v.x, -v.y); }
#pragma unroll
        for (int r = 0; r < W; ++r) {
          cplx v = tile[r * PC_NT];
#pragma unroll
          for (int c = 0; c < W; ++c) cfma(v, __ldg(Ck + r * W + c), xs[c]);
          tile[r * PC_NT] = v;
        }
      }
      if (q + 1 < p.P) {
        const cplx* ys = p.y + (size_t)p.phi[q] * ld + a;
#pragma unroll
        for (int c = 0; c < W; ++c) { const cplx v = ys[(size_t)c * ld]; xs[c] = make_double2(-v.x, -v.y); }
#pragma unroll
        for (int r = 0; r < W; ++r) {
          cplx v = tile[(n_rad - W + r) * PC_NT];
#pragma unroll
          for (int c = 0; c < W; ++c) cfma(v, __ldg(Ck + WW + r * W + c), xs[c]);
          tile[(n_rad - W + r) * PC_NT] = v;
        }
      }
    }
#pragma unroll
    for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
    for (int s = 0; s < nst; ++s) {
      const int r0 = s * PC_ROWS, nr = min(PC_ROWS, n_rad - r0);
      issue(s + PC_STAGES - 1);
      cp_async_wait<PC_STAGES - 1>();
      __syncwarp();
      const cplx* cs = ring + (size_t)(s % PC_STAGES) * PL::STAGE + (size_t)(slot >= 0 ? slot : 0) * PC_ROWS * PL::CW;
      const cplx* cg = p.Lcol + ((size_t)k * n_tot + row0 + r0) * W;
      cplx xc[PC_ROWS];
#pragma unroll
      for (int r = 0; r < PC_ROWS; ++r) xc[r] = tile[min(r0 + r, n_rad - 1) * PC_NT];
#pragma unroll
      for (int r = 0; r < PC_ROWS; ++r) {
        if (r < nr) {
          const cplx xi = xc[r];
          cplx c[W];
          if (slot >= 0) {
#pragma unroll
            for (int d = 0; d < W; ++d) c[d] = cs[r * W + d];
          } else {
#pragma unroll
            for (int d = 0; d < W; ++d) c[d] = __ldg(cg + r * W + d);
          }
          const cplx nc0 = make_double2(-c[0].x, -c[0].y);
          cplx base = pw[1];
          cfma(base, nc0, xi);                                       // off the chain
          const cplx yi = cadd(xi, pw[0]);
          tile[(r0 + r) * PC_NT] = yi;
          const cplx nyi = make_double2(-yi.x, -yi.y);
          cfma(base, nc0, pw[0]);                                    // the chain: one complex FMA per row
          pw[0] = base;
#pragma unroll
          for (int d = 1; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], c[d], nyi); }
        }
      }
      __syncwarp();
    }
    cp_async_wait<0>();
  }
  // ================= backward: U x = y (rows descending; stage s covers rows [n_rad - (s+1) R, n_rad - s R)) ====
  {
    auto issue = [&](int s) {
      if (s < nst) {
        cplx* st = ring + (size_t)(s % PC_STAGES) * PL::STAGE;
        const int hi = n_rad - s * PC_ROWS, lo = max(0, hi - PC_ROWS), nr = hi - lo;
        for (int c = 0; c < ncls; ++c) {
          const cplx* src = p.Ucol + ((size_t)wcls[c] * n_tot + row0 + lo) * (W + 1);
          cplx* dst = st + (size_t)c * PC_ROWS * PL::CW;
          for (int e = lane; e < nr * (W + 1); e += PC_NT) cp_async16(dst + e, src + e);
        }
      }
      cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
    for (int s = 0; s < PC_STAGES - 1; ++s) issue(s);
    for (int s = 0; s < nst; ++s) {
      const int hi = n_rad - s * PC_ROWS, lo = max(0, hi - PC_ROWS), nr = hi - lo;
      issue(s + PC_STAGES - 1);
      cp_async_wait<PC_STAGES - 1>();
      __syncwarp();
      const cplx* cs = ring + (size_t)(s % PC_STAGES) * PL::STAGE + (size_t)(slot >= 0 ? slot : 0) * PC_ROWS * PL::CW;
      const cplx* cg = p.Ucol + ((size_t)k * n_tot + row0 + lo) * (W + 1);
      cplx xc[PC_ROWS];                                              // xc[rr] = row hi - 1 - rr: the order of consumption
#pragma unroll
      for (int rr = 0; rr < PC_ROWS; ++rr) xc[rr] = tile[max(hi - 1 - rr, 0) * PC_NT];
#pragma unroll
      for (int rr = 0; rr < PC_ROWS; ++rr) {
        if (rr < nr) {
          const int r = nr - 1 - rr;                                 // row lo + r, factor row r of the stage
          const cplx yi = xc[rr];
          cplx c[W + 1];
          if (slot >= 0) {
#pragma unroll
            for (int d = 0; d <= W; ++d) c[d] = cs[r * (W + 1) + d];
          } else {
#pragma unroll
            for (int d = 0; d <= W; ++d) c[d] = __ldg(cg + r * (W + 1) + d);
          }
          // x_i = uinv (y_i + pw0);  pw0' = pw1 - U[i-1][i] x_i = (pw1 - c1 y_i) - c1 pw0  with c1 = U[i-1][i] uinv
          const cplx nc1 = make_double2(-c[1].x, -c[1].y);
          cplx base = pw[1];
          cfma(base, nc1, yi);                                       // off the chain
          const cplx xi = cmul(cadd(yi, pw[0]), c[0]);
          yout[(size_t)(lo + r) * ld] = xi;
          const cplx nxi = make_double2(-xi.x, -xi.y);
          cfma(base, nc1, pw[0]);                                    // the chain
          pw[0] = base;
#pragma unroll
          for (int d = 1; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], c[d + 1], nxi); }
        }
      }
      __syncwarp();
    }
    cp_async_wait<0>();
  }
}

// runtime-w fallback (13 < w <= 32): two plain sweeps through global memory, one thread per channel
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
    const cplx t = cadd(p.y[(size_t)i * ld + a], pw[0]);
    const cplx xi = cmul(t, uc[0]);
    p.y[(size_t)i * ld + a] = xi;
    const cplx nxi = make_double2(-xi.x, -xi.y);
    // Ucol[.][1] is pre-scaled by 1/U[i][i]: it multiplies (y_i + pw0), not x_i
    if (W >= 1) { pw[0] = pw[1]; cfma(pw[0], uc[1], make_double2(-t.x, -t.y)); }
    for (int d = 1; d < W; ++d) { pw[d] = pw[d + 1]; cfma(pw[d], uc[d + 1], nxi); }
  }
}

template <int W>
static int launch_precond_w(const PrecArgs& a, cudaStream_t s) {
  const size_t smem = PrecPlan<W>::smem(a.tile_rows);
  if (cudaFuncSetAttribute(k_precond_tile<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
  int n = 0;
  if (a.P > 1) {
    k_precond_spikes<W><<<dim3((a.ld + 127) / 128, a.P), 128, 0, s>>>(a);
    k_precond_schur<W><<<a.ld / PC_NT, PC_NT, 0, s>>>(a);
    n = 2;
  }
  k_precond_tile<W><<<dim3(a.ld / PC_NT, a.P), PC_NT, smem, s>>>(a);
  return n + 1;
}

size_t precond_tile_smem(int w, int tile_rows) {
  return ((size_t)PC_STAGES * PC_MAXC * PC_ROWS * (w + 1) + (size_t)tile_rows * PC_NT) * sizeof(cplx);
}

int launch_precond(const PrecArgs& a, cudaStream_t s) {
  switch (a.w) {
#define X(W) case W: return launch_precond_w<W>(a, s);
    TDDE_PC_WIDTHS(X)
#undef X
    default:
      if (a.w > 32 || a.w < 1 || a.P != 1) return -1;
      k_precond_any<<<(a.ld + PC_NT - 1) / PC_NT, PC_NT, 0, s>>>(a);
  }
  return 1;
}
