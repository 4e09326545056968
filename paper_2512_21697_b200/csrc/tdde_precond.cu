// tdde_precond.cu -- y = (S + i dt/2 H0)^{-1} x as batched banded solves (
// PAPER.md:211-215, Eq. 26: M is block-diagonal over angular channels, LU factors computed at start-up).
//
// The radial index is cut into P interiors separated by P-1 separators of w rows (tdde_partition.h); the solve is an
// exact reordering of Gaussian elimination in three kernels:
//   P1  k_precond_spikes   r(-)_q, r(+)_q = W b_I : streaming, 2 w complex FMAs per interior row, one read of b
//   P2  k_precond_schur    block-Thomas solve of the block-tridiagonal Schur system for the separator unknowns
//   P2b k_precond_corners  A_IS x_S for the first / last w rows of every interior (tiny, fully parallel)
//   P3  k_precond_tile     per (32 channels x interior): b_I - A_IS x_S into a SHARED-MEMORY tile, L sweep and U sweep on
//                          the tile, one coalesced write of x_I.  No intermediate vector ever goes to global memory.
// Algorithmic traffic: 16 B (P1) + 32 B (P3) per element instead of 96 B for sweep / store / reload / correct.
// One warp per 32 consecutive channels, lane = channel (coalesced 16-byte accesses in the internal layout).  Both
// sweeps run in column-oriented (axpy) form: once y_i is final the W pending rows below it are updated independently;
// only the update of the next row is on the critical path, and it is split as  pw0' = (pw1 - c x_i) - c pw0  so that
// the chain is short; for the U sweep the host pre-scales U[i-1][i] by 1/U[i][i] for the same reason.  Factor rows of
// the (few) kappa-classes present in the warp stream through a cp.async ring in shared memory; inside a stage the operands
// of the next row are loaded into registers before the arithmetic of the current one.
// Factor layout (tdde_partition.cu): Lcol[k][i][d-1] = L[i+d][i];
//   Ucol[k][i][0] = 1/U[i][i], Ucol[k][i][1] = U[i-1][i] / U[i][i], Ucol[k][i][d>=2] = U[i-d][i].
#include "tdde_reduce.cuh"

#define PC_NT 32
// Schur chain, W > 8: the block rows do not fit a second register set, so they are prefetched into L1 (prefetch.global.L1) four steps
// ahead and read at use, and only b, m1, m2 (resp. z) are held per set (bandwidth 19: solve 0.895 -> 0.844 ms).  W <= 8 keeps two full
// register sets: the same scheme measured slower there (HBM-scale W = 6: 0.504 -> 0.540 ms).
#ifndef TDDE_SCHUR_L1PF
#define TDDE_SCHUR_L1PF(W) ((W) > 8)
#endif
#ifndef TDDE_SCHUR_DEPTH
#define TDDE_SCHUR_DEPTH(W) (TDDE_SCHUR_L1PF(W) ? 4 : 2)   // full sets: 3 and 4 spill and lose (HBM-scale solve 0.50 -> 0.56 / 0.60 ms)
#endif
#define PC_ROWS 8
#ifndef PC_STAGES
#define PC_STAGES 2
#endif
#define PC_MAXC TDDE_PC_MAXC

template <int W>
struct PrecPlan {
  static constexpr int CW = W + 1;                                   // coefficient row width (U needs W+1)
  static constexpr int STAGE = PC_MAXC * PC_ROWS * CW;               // complex per stage (factor rows only)
  static constexpr int RING = PC_STAGES * STAGE;                     // complex
  static size_t smem(int tile_rows) { return ((size_t)RING + (size_t)tile_rows * PC_NT) * sizeof(cplx); }
};

// ---- P1: spike dot products.  CTA = 128 channels x one interior; thread = channel.  The spike rows of the CTA's
// kappa-classes (the class lists of the operator apply: <= TDDE_AP_MAXC per 128 channels) are staged in shared memory in
// chunks of SPK_ROWS rows with cp.async, double-buffered, and read back as (mostly) warp-broadcasts. ----
#define SPK_ROWS 8
template <int W>
__global__ void __launch_bounds__(128) k_precond_spikes(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* Ws = reinterpret_cast<cplx*>(smem_raw);                      // [2][TDDE_AP_MAXC][SPK_ROWS][2W]
  constexpr int CH = SPK_ROWS * 2 * W;                               // complex per class per chunk
  const int tid = threadIdx.x, ld = p.ld;
  const int a = blockIdx.x * 128 + tid;
  const bool ok = a < ld;
  const int ac = ok ? a : ld - 1;
  const int q = blockIdx.y;
  const int lo = pc_lo(p, q), len = pc_len(p, q);
  const int* ccls = p.cta_cls + blockIdx.x * TDDE_AP_MAXC;
  int ncls = 0;
#pragma unroll
  for (int c = 0; c < TDDE_AP_MAXC; ++c) ncls += (ccls[c] >= 0);
  const int slot = p.aslot[ac];
  const cplx* Wg = p.Wsp + ((size_t)p.cls[ac] * p.n_rad + lo) * 2 * W;     // global fallback (class not staged)
  const int nch = (len + SPK_ROWS - 1) / SPK_ROWS;
  auto issue = [&](int c) {
    if (c < nch) {
      const int r0 = c * SPK_ROWS, nr = min(SPK_ROWS, len - r0);
      cplx* dst0 = Ws + (size_t)(c & 1) * TDDE_AP_MAXC * CH;
      for (int s = 0; s < ncls; ++s) {
        const cplx* src = p.Wsp + ((size_t)ccls[s] * p.n_rad + lo + r0) * 2 * W;
        for (int e = tid; e < nr * 2 * W; e += 128) cp_async16(dst0 + s * CH + e, src + e);
      }
    }
    cp_async_commit();
  };
  issue(0);
  const cplx* xin = p.x + (size_t)lo * ld + ac;
  cplx am[W], ap[W];
#pragma unroll
  for (int c = 0; c < W; ++c) am[c] = ap[c] = make_double2(0, 0);
  cplx bn[SPK_ROWS];
#pragma unroll
  for (int r = 0; r < SPK_ROWS; ++r) bn[r] = (r < len) ? xin[(size_t)r * ld] : make_double2(0, 0);
  for (int c = 0; c < nch; ++c) {
    const int r0 = c * SPK_ROWS, nr = min(SPK_ROWS, len - r0);
    cplx b[SPK_ROWS];
#pragma unroll
    for (int r = 0; r < SPK_ROWS; ++r) b[r] = bn[r];
    issue(c + 1);
#pragma unroll
    for (int r = 0; r < SPK_ROWS; ++r) bn[r] = (r0 + SPK_ROWS + r < len) ? xin[(size_t)(r0 + SPK_ROWS + r) * ld] : make_double2(0, 0);
    cp_async_wait<1>();
    __syncthreads();
    const cplx* wl = Ws + (size_t)(c & 1) * TDDE_AP_MAXC * CH + (size_t)(slot >= 0 ? slot : 0) * CH;
    if (slot >= 0) {
#pragma unroll
      for (int r = 0; r < SPK_ROWS; ++r) {
        if (r < nr) {
#pragma unroll
          for (int e = 0; e < W; ++e) { cfma(am[e], wl[r * 2 * W + e], b[r]); cfma(ap[e], wl[r * 2 * W + W + e], b[r]); }
        }
      }
    } else {
      for (int r = 0; r < nr; ++r) {
        const cplx* wr = Wg + (size_t)(r0 + r) * 2 * W;
#pragma unroll
        for (int e = 0; e < W; ++e) { cfma(am[e], __ldg(wr + e), b[r]); cfma(ap[e], __ldg(wr + W + e), b[r]); }
      }
    }
    __syncthreads();                                                  // the other buffer may be overwritten next round
  }
  cp_async_wait<0>();
  if (ok) {
#pragma unroll
    for (int c = 0; c < W; ++c) {
      p.rsm[((size_t)q * W + c) * ld + a] = am[c];
      p.rsp[((size_t)q * W + c) * ld + a] = ap[c];
    }
  }
}

// ---- P1 fused into the BiCGSTAB vector updates that PRODUCE the right-hand side of the solve: the p-update
// (MODE 0: p = r + beta (p - omega v), first iteration p = r) or the s-update (MODE 1: s = r - alpha v with ||s||^2) runs on a
// (128 channels x interior) decomposition and forms the spike dot products of the vector it has just computed, so the solve
// never re-reads its right-hand side for them.  CTA (bx, q) also updates the separator rows after interior q. ----
#define VSP_ROWS 4
template <int W, int MODE>
__global__ void __launch_bounds__(128) k_vec_spikes(const VecArgs v, const PrecArgs p) {
  const SolverState* st = v.red.st;
  if (solver_idle(st)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* Ws = reinterpret_cast<cplx*>(smem_raw);                      // [2][TDDE_AP_MAXC][VSP_ROWS][2W]
  constexpr int CH = VSP_ROWS * 2 * W;
  const int tid = threadIdx.x, ld = p.ld;
  const int a = blockIdx.x * 128 + tid;
  const bool ok = a < ld;
  const int ac = ok ? a : ld - 1;
  const int q = blockIdx.y;
  const int lo = pc_lo(p, q), len = pc_len(p, q);
  const int nrows = len + (q + 1 < p.P ? W : 0);                     // interior + the separator after it
  const int* ccls = p.cta_cls + blockIdx.x * TDDE_AP_MAXC;
  int ncls = 0;
#pragma unroll
  for (int c = 0; c < TDDE_AP_MAXC; ++c) ncls += (ccls[c] >= 0);
  const int slot = p.aslot[ac];
  const cplx* Wg = p.Wsp + ((size_t)p.cls[ac] * p.n_rad + lo) * 2 * W;
  const int nch = (nrows + VSP_ROWS - 1) / VSP_ROWS;
  auto issue = [&](int c) {
    const int r0 = c * VSP_ROWS, nr = min(VSP_ROWS, len - r0);       // spike rows exist for interior rows only
    if (nr > 0) {
      cplx* dst0 = Ws + (size_t)(c & 1) * TDDE_AP_MAXC * CH;
      for (int s = 0; s < ncls; ++s) {
        const cplx* src = p.Wsp + ((size_t)ccls[s] * p.n_rad + lo + r0) * 2 * W;
        for (int e = tid; e < nr * 2 * W; e += 128) cp_async16(dst0 + s * CH + e, src + e);
      }
    }
    cp_async_commit();
  };
  const bool first = st->first;
  const cplx beta = st->beta, omega = st->omega, alpha = st->alpha;
  const size_t base = (size_t)lo * ld + ac;
  const cplx *rin = v.r + base, *vin = v.v + base;
  cplx* pio = (MODE == 0 ? v.p : v.s) + base;
  cplx rn[VSP_ROWS], vn[VSP_ROWS], pn[VSP_ROWS];
  auto fetch = [&](int c) {
    const int r0 = c * VSP_ROWS;
#pragma unroll
    for (int r = 0; r < VSP_ROWS; ++r) {
      const bool in = r0 + r < nrows;
      rn[r] = in ? rin[(size_t)(r0 + r) * ld] : make_double2(0, 0);
      if (MODE == 1 || !first) vn[r] = in ? vin[(size_t)(r0 + r) * ld] : make_double2(0, 0);
      if (MODE == 0 && !first) pn[r] = in ? pio[(size_t)(r0 + r) * ld] : make_double2(0, 0);
    }
  };
  issue(0);
  fetch(0);
  cplx am[W], ap[W];
#pragma unroll
  for (int c = 0; c < W; ++c) am[c] = ap[c] = make_double2(0, 0);
  double s2 = 0;
  for (int c = 0; c < nch; ++c) {
    const int r0 = c * VSP_ROWS, nr = min(VSP_ROWS, nrows - r0), nri = min(VSP_ROWS, len - r0);
    cplx b[VSP_ROWS];
#pragma unroll
    for (int r = 0; r < VSP_ROWS; ++r) {
      if (MODE == 0) {
        b[r] = rn[r];
        if (!first) {
          cplx t = pn[r];
          cfms(t, omega, vn[r]);                                     // p - omega v
          cfma(b[r], beta, t);
        }
      } else {
        b[r] = rn[r];
        cfms(b[r], alpha, vn[r]);
        if (r < nr && ok) { s2 = fma(b[r].x, b[r].x, s2); s2 = fma(b[r].y, b[r].y, s2); }
      }
    }
    issue(c + 1);
    if (c + 1 < nch) fetch(c + 1);
    if (ok) {
#pragma unroll
      for (int r = 0; r < VSP_ROWS; ++r)
        if (r < nr) pio[(size_t)(r0 + r) * ld] = b[r];
    }
    cp_async_wait<1>();
    __syncthreads();
    if (nri > 0) {
      const cplx* wl = Ws + (size_t)(c & 1) * TDDE_AP_MAXC * CH + (size_t)(slot >= 0 ? slot : 0) * CH;
      if (slot >= 0) {
#pragma unroll
        for (int r = 0; r < VSP_ROWS; ++r) {
          if (r < nri) {
#pragma unroll
            for (int e = 0; e < W; ++e) { cfma(am[e], wl[r * 2 * W + e], b[r]); cfma(ap[e], wl[r * 2 * W + W + e], b[r]); }
          }
        }
      } else {
        for (int r = 0; r < nri; ++r) {
          const cplx* wr = Wg + (size_t)(r0 + r) * 2 * W;
#pragma unroll
          for (int e = 0; e < W; ++e) { cfma(am[e], __ldg(wr + e), b[r]); cfma(ap[e], __ldg(wr + W + e), b[r]); }
        }
      }
    }
    __syncthreads();
  }
  cp_async_wait<0>();
  if (ok) {
#pragma unroll
    for (int c = 0; c < W; ++c) {
      p.rsm[((size_t)q * W + c) * ld + a] = am[c];
      p.rsp[((size_t)q * W + c) * ld + a] = ap[c];
    }
  }
  if (MODE == 1) grid_reduce_finalize<128>(0.0, 0.0, s2, v.red);
}

// ---- P2: block Thomas over the separators.  CTA = 32 channels x W warps; warp c owns row c of every w x w block product,
// lane = channel.  r_j = b_S(j) - r(+)_j - r(-)_{j+1};
//   forward   r'_j = r_j - (B_j D'^-1_{j-1}) r'_{j-1},  z_j = D'^-1_j r'_j   (z_j kept in the r(+) scratch)
//   backward  x_j = z_j - (D'^-1_j C_j) x_{j+1}
// one CTA barrier per step.  Software pipelining: the operands of the next step are loaded, untouched, into a second register
// set before the block products of the current step (loops unrolled by two so the sets swap roles without copies). ----
template <int W>
struct SchurFwd { cplx b, m1, m2, lb[TDDE_SCHUR_L1PF(W) ? 1 : W], di[TDDE_SCHUR_L1PF(W) ? 1 : W]; };
template <int W>
struct SchurBwd { cplx z, g[TDDE_SCHUR_L1PF(W) ? 1 : W]; };
__device__ __forceinline__ void pf_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

template <int W>
__global__ void __launch_bounds__(PC_NT* W, (W <= 6 ? 2 : 1)) k_precond_schur(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  __shared__ cplx sh[2][W][PC_NT];
  const int lane = threadIdx.x & 31, c = threadIdx.x >> 5;
  const int a = blockIdx.x * PC_NT + lane;
  const int ld = p.ld, ns = p.P - 1;
  constexpr int WW = W * W;
  const cplx* Sk = p.Schur + (size_t)p.cls[a] * ns * 3 * WW + c * W;  // row c of every block
  auto sep_row = [&](int j) { return pc_lo(p, j) + pc_len(p, j) + c; };
  constexpr bool L1PF = TDDE_SCHUR_L1PF(W);
  constexpr int D = TDDE_SCHUR_DEPTH(W);    // operand sets in flight: each is 2 W + 3 complex registers in the forward pass
  // ---------------- forward ----------------
  auto ffetch = [&](int j, SchurFwd<W>& o) {
    if (j >= ns) return;
    o.b = p.x[(size_t)sep_row(j) * ld + a];
    o.m1 = p.rsp[((size_t)j * W + c) * ld + a];
    o.m2 = p.rsm[((size_t)(j + 1) * W + c) * ld + a];
    const cplx* rb = Sk + (size_t)j * 3 * WW;                       // rows c of B_j D'^-1_{j-1} and of D'^-1_j: W x 16 bytes each
    if (L1PF) { pf_l1(rb); pf_l1(rb + W - 1); pf_l1(rb + WW); pf_l1(rb + WW + W - 1); }
    else {
#pragma unroll
      for (int q = 0; q < (L1PF ? 1 : W); ++q) { o.lb[q] = __ldg(rb + q); o.di[q] = __ldg(rb + WW + q); }
    }
  };
  // r'_{j-1} is in sh[(j-1) & 1]; publishes r'_j in sh[j & 1], then row c of z_j
#define LB(q) (L1PF ? __ldg(Sk + (size_t)j * 3 * WW + (q)) : o.lb[L1PF ? 0 : (q)])
#define DI(q) (L1PF ? __ldg(Sk + (size_t)j * 3 * WW + WW + (q)) : o.di[L1PF ? 0 : (q)])
#define GG(q) (L1PF ? __ldg(Sk + (size_t)j * 3 * WW + 2 * WW + (q)) : o.g[L1PF ? 0 : (q)])
  auto fstep = [&](int j, const SchurFwd<W>& o) {
    cplx r0 = make_double2(o.b.x - o.m1.x - o.m2.x, o.b.y - o.m1.y - o.m2.y), r1 = make_double2(0, 0);
    if (j > 0) {
#pragma unroll
      for (int q = 0; q < W; q += 2) {
        cfms(r0, LB(q), sh[(j - 1) & 1][q][lane]);
        if (q + 1 < W) cfms(r1, LB(q + 1), sh[(j - 1) & 1][q + 1][lane]);
      }
    }
    sh[j & 1][c][lane] = cadd(r0, r1);
    __syncthreads();
    cplx z0 = make_double2(0, 0), z1 = make_double2(0, 0);
#pragma unroll
    for (int q = 0; q < W; q += 2) {
      cfma(z0, DI(q), sh[j & 1][q][lane]);
      if (q + 1 < W) cfma(z1, DI(q + 1), sh[j & 1][q + 1][lane]);
    }
    p.rsp[((size_t)j * W + c) * ld + a] = cadd(z0, z1);
  };
  // operands of step j + D - 1 are requested before step j runs: the chain is latency-bound (one block product and one CTA barrier
  // per step), so the loads of D - 1 steps are in flight behind it
  {
    SchurFwd<W> buf[D];
#pragma unroll
    for (int k = 0; k < D - 1; ++k) ffetch(k, buf[k]);
    for (int j = 0; j < ns; j += D) {
#pragma unroll
      for (int k = 0; k < D; ++k) {
        if (j + k < ns) {
          ffetch(j + k + D - 1, buf[(k + D - 1) % D]);
          fstep(j + k, buf[k]);
        }
      }
    }
  }
  __syncthreads();
  // ---------------- backward: x_{j+1} is in sh[(j+1) & 1] ----------------
  auto bfetch = [&](int j, SchurBwd<W>& o) {
    if (j < 0) return;
    o.z = p.rsp[((size_t)j * W + c) * ld + a];
    if (L1PF) { pf_l1(Sk + (size_t)j * 3 * WW + 2 * WW); pf_l1(Sk + (size_t)j * 3 * WW + 2 * WW + W - 1); }
    else {
#pragma unroll
      for (int q = 0; q < (L1PF ? 1 : W); ++q) o.g[q] = __ldg(Sk + (size_t)j * 3 * WW + 2 * WW + q);
    }
  };
  auto bstep = [&](int j, const SchurBwd<W>& o) {
    cplx x0 = o.z, x1 = make_double2(0, 0);
    if (j + 1 < ns) {
#pragma unroll
      for (int q = 0; q < W; q += 2) {
        cfms(x0, GG(q), sh[(j + 1) & 1][q][lane]);
        if (q + 1 < W) cfms(x1, GG(q + 1), sh[(j + 1) & 1][q + 1][lane]);
      }
    }
    const cplx xv = cadd(x0, x1);
    p.y[(size_t)sep_row(j) * ld + a] = xv;
    sh[j & 1][c][lane] = xv;
    __syncthreads();
  };
  {
    SchurBwd<W> buf[D];
#pragma unroll
    for (int k = 0; k < D - 1; ++k) bfetch(ns - 1 - k, buf[k]);
    for (int j = ns - 1; j >= 0; j -= D) {
#pragma unroll
      for (int k = 0; k < D; ++k) {
        if (j - k >= 0) {
          bfetch(j - k - (D - 1), buf[(k + D - 1) % D]);
          bstep(j - k, buf[k]);
        }
      }
    }
  }
}

#undef LB
#undef DI
#undef GG

// ---- P2b: with every x_S known, A_IS x_S for the interiors next to each separator: the last w rows of interior j (into r(+)_j)
// and the first w rows of interior j+1 (into r(-)_{j+1}).  One thread per (separator, channel). ----
template <int W>
__global__ void __launch_bounds__(128) k_precond_corners(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * 128 + threadIdx.x;
  if (a >= p.ld) return;
  const int j = blockIdx.y, ld = p.ld;                               // one thread per (separator, channel): x_S loaded once
  constexpr int WW = W * W;
  const cplx* Ck = p.Corner + (size_t)p.cls[a] * p.P * 2 * WW;
  const cplx* tT = Ck + ((size_t)(j + 1) * 2 + 0) * WW;               // top corner of interior j + 1
  const cplx* tB = Ck + ((size_t)j * 2 + 1) * WW;                     // bottom corner of interior j
  const cplx* xs = p.y + (size_t)(pc_lo(p, j) + pc_len(p, j)) * ld + a;
  cplx xv[W];
#pragma unroll
  for (int q = 0; q < W; ++q) xv[q] = xs[(size_t)q * ld];
#pragma unroll
  for (int c = 0; c < W; ++c) {
    cplx ct = make_double2(0, 0), cb = make_double2(0, 0);
#pragma unroll
    for (int q = 0; q < W; ++q) {
      cfma(ct, __ldg(tT + c * W + q), xv[q]);
      cfma(cb, __ldg(tB + c * W + q), xv[q]);
    }
    p.rsm[((size_t)(j + 1) * W + c) * ld + a] = ct;
    p.rsp[((size_t)j * W + c) * ld + a] = cb;
  }
}

// ---- P3: one warp = 32 channels x one interior.  The right-hand side lives in a shared-memory tile (one column per lane, so
// no inter-lane hazards) from its load to the end of the U sweep; factor rows of the warp's kappa-classes stream through a
// cp.async ring.  STAGED: every lane's class is in the ring (warp-uniform fast path); otherwise coefficients come from global. ----
// Column-oriented (axpy) sweeps with explicit software pipelining: the factor row and the tile element of row r + 1 are
// loaded into a second register set before the arithmetic of row r (a warp issues in order, so a load placed next to its
// use costs its full latency on every row).  Once y_i is final the W pending rows below it are updated independently; only
// the update of the next row is on the critical path, split as  pw0' = (pw1 - c x_i) - c pw0.
template <int W, bool STAGED>
__device__ __forceinline__ void pc_l_rows(const cplx* __restrict__ cs, const cplx* __restrict__ cg, cplx* trow, int nr, cplx (&pw)[W + 1]) {
  cplx cn[W], xn;
  auto load = [&](int r, cplx (&c)[W], cplx& x) {
    x = trow[r * PC_NT];
#pragma unroll
    for (int d = 0; d < W; ++d) c[d] = STAGED ? cs[r * W + d] : __ldg(cg + r * W + d);
  };
  load(0, cn, xn);
#pragma unroll
  for (int r = 0; r < PC_ROWS; ++r) {
    if (r < nr) {
      cplx c[W];
      const cplx xi = xn;
#pragma unroll
      for (int d = 0; d < W; ++d) c[d] = cn[d];
      if (r + 1 < PC_ROWS && r + 1 < nr) load(r + 1, cn, xn);
      cplx base = pw[1];
      cfms(base, c[0], xi);                                          // off the chain
      const cplx yi = cadd(xi, pw[0]);
      trow[r * PC_NT] = yi;
      cfms(base, c[0], pw[0]);                                       // the chain: one complex FMA per row
      pw[0] = base;
#pragma unroll
      for (int d = 1; d < W; ++d) { pw[d] = pw[d + 1]; cfms(pw[d], c[d], yi); }
    }
  }
}
template <int W, bool STAGED>
__device__ __forceinline__ void pc_u_rows(const cplx* __restrict__ cs, const cplx* __restrict__ cg, const cplx* trow, cplx* yrow, size_t ld, int nr,
                                          cplx (&pw)[W + 1]) {
  // trow / yrow point at row `lo` of the stage; rows are consumed from lo + nr - 1 down to lo
  cplx cn[W + 1], yn;
  auto load = [&](int r, cplx (&c)[W + 1], cplx& y) {
    y = trow[r * PC_NT];
#pragma unroll
    for (int d = 0; d <= W; ++d) c[d] = STAGED ? cs[r * (W + 1) + d] : __ldg(cg + r * (W + 1) + d);
  };
  load(nr - 1, cn, yn);
#pragma unroll
  for (int rr = 0; rr < PC_ROWS; ++rr) {
    const int r = nr - 1 - rr;
    if (r >= 0) {
      cplx c[W + 1];
      const cplx yi = yn;
#pragma unroll
      for (int d = 0; d <= W; ++d) c[d] = cn[d];
      if (r > 0) load(r - 1, cn, yn);
      // x_i = uinv (y_i + pw0);  pw0' = pw1 - U[i-1][i] x_i = (pw1 - c1 y_i) - c1 pw0  with c1 = U[i-1][i] uinv
      cplx base = pw[1];
      cfms(base, c[1], yi);                                          // off the chain
      const cplx xi = cmul(cadd(yi, pw[0]), c[0]);
      yrow[(size_t)r * ld] = xi;
      cfms(base, c[1], pw[0]);                                       // the chain
      pw[0] = base;
#pragma unroll
      for (int d = 1; d < W; ++d) { pw[d] = pw[d + 1]; cfms(pw[d], c[d + 1], xi); }
    }
  }
}

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
  const int row0 = pc_lo(p, q);
  const int n_rad = pc_len(p, q);                                 // rows of this interior
  const cplx* xin = p.x + (size_t)row0 * ld + a;
  cplx* yout = p.y + (size_t)row0 * ld + a;
  const int* wcls = p.warp_cls + blockIdx.x * PC_MAXC;
  int ncls = 0;
#pragma unroll
  for (int c = 0; c < PC_MAXC; ++c) ncls += (wcls[c] >= 0);
  const int slot = p.slot[a];
  const bool staged = __all_sync(0xffffffffu, slot >= 0);
  const int k = p.cls[a];
  const int nst = (n_rad + PC_ROWS - 1) / PC_ROWS;
  const int tail = n_rad - (nst - 1) * PC_ROWS;                      // rows of the last (forward) / first-consumed (backward) stage

  // right-hand side rows -> tile (asynchronous, all rows in flight at once)
  {
    const cplx* src = xin;
    cplx* dst = tile;
    for (int r = 0; r < n_rad; ++r) { cp_async16(dst, src); dst += PC_NT; src += ld; }
  }
  cp_async_commit();

  cplx pw[W + 1];
  // One stage sequence for both sweeps: stages 0 .. nst-1 are the L rows top-down, stages nst .. 2 nst-1 the U rows bottom-up
  // (the ragged stage first, so all later ones are full).  Stage t + PC_STAGES - 1 is requested while stage t is consumed.
  auto issue = [&](int t) {
    if (staged && t < 2 * nst) {
      const bool up = t >= nst;
      const int s = up ? t - nst : t;
      const int first_row = up ? (nst - 1 - s) * PC_ROWS : s * PC_ROWS;
      const int nr = (up ? s == 0 : s == nst - 1) ? tail : PC_ROWS;
      const int cw = up ? W + 1 : W;
      const cplx* fac = up ? p.Ucol : p.Lcol;
      cplx* st = ring + (size_t)(t % PC_STAGES) * PL::STAGE;
      for (int c = 0; c < ncls; ++c) {
        const cplx* src = fac + ((size_t)wcls[c] * n_tot + row0 + first_row) * cw;
        cplx* dst = st + (size_t)c * PC_ROWS * PL::CW;
        for (int e = lane; e < nr * cw; e += PC_NT) cp_async16(dst + e, src + e);
      }
    }
    cp_async_commit();
  };
  for (int t = 0; t < PC_STAGES - 1; ++t) issue(t);

  // A_IS x_S for the first / last w rows (formed by k_precond_schur): loads first, then the wait for the tile
  if (p.P > 1) {
    const bool has_m = q > 0, has_p = q + 1 < p.P;
    cplx cm[W], cp[W];
#pragma unroll
    for (int c = 0; c < W; ++c) {
      cm[c] = has_m ? p.rsm[((size_t)q * W + c) * ld + a] : make_double2(0, 0);
      cp[c] = has_p ? p.rsp[((size_t)q * W + c) * ld + a] : make_double2(0, 0);
    }
    cp_async_wait<PC_STAGES - 1>();                                  // the tile has landed (own column: no warp sync needed)
    cplx* tb = tile + (n_rad - W) * PC_NT;
#pragma unroll
    for (int r = 0; r < W; ++r) { const cplx v = tile[r * PC_NT]; tile[r * PC_NT] = csub(v, cm[r]); }
#pragma unroll
    for (int r = 0; r < W; ++r) { const cplx v = tb[r * PC_NT]; tb[r * PC_NT] = csub(v, cp[r]); }
  }
  // ================= forward: L y = b_I - A_IS x_S =================
#pragma unroll
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
  {
    const cplx* cg = p.Lcol + ((size_t)k * n_tot + row0) * W;
    for (int s = 0; s < nst; ++s) {
      const int nr = (s + 1 < nst) ? PC_ROWS : tail;
      issue(s + PC_STAGES - 1);
      cp_async_wait<PC_STAGES - 1>();
      __syncwarp();
      const cplx* cs = ring + (size_t)(s % PC_STAGES) * PL::STAGE + (size_t)(staged ? slot : 0) * PC_ROWS * PL::CW;
      cplx* trow = tile + s * PC_ROWS * PC_NT;
      if (staged) {
        if (nr == PC_ROWS) pc_l_rows<W, true>(cs, cg, trow, PC_ROWS, pw);
        else pc_l_rows<W, true>(cs, cg, trow, nr, pw);
      } else {
        pc_l_rows<W, false>(cs, cg + (size_t)s * PC_ROWS * W, trow, nr, pw);
      }
      __syncwarp();
    }
  }
  // ================= backward: U x = y, rows descending =================
#pragma unroll
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
  {
    const cplx* cg = p.Ucol + ((size_t)k * n_tot + row0) * (W + 1);
    for (int s = 0; s < nst; ++s) {
      const int lo = (nst - 1 - s) * PC_ROWS, nr = s == 0 ? tail : PC_ROWS;
      issue(nst + s + PC_STAGES - 1);
      cp_async_wait<PC_STAGES - 1>();
      __syncwarp();
      const cplx* cs = ring + (size_t)((nst + s) % PC_STAGES) * PL::STAGE + (size_t)(staged ? slot : 0) * PC_ROWS * PL::CW;
      const cplx* trow = tile + lo * PC_NT;
      cplx* yrow = yout + (size_t)lo * ld;
      if (staged) {
        if (nr == PC_ROWS) pc_u_rows<W, true>(cs, cg, trow, yrow, ld, PC_ROWS, pw);
        else pc_u_rows<W, true>(cs, cg, trow, yrow, ld, nr, pw);
      } else {
        pc_u_rows<W, false>(cs, cg + (size_t)lo * (W + 1), trow, yrow, ld, nr, pw);
      }
      __syncwarp();
    }
  }
  cp_async_wait<0>();
}

// runtime-w fallback (13 < w <= 32): pending rows in a small local array, direct global loads, one thread per channel
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
    for (int d = 0; d < W; ++d) { pw[d] = pw[d + 1]; cfms(pw[d], Lc[(size_t)i * W + d], yi); }
  }
  for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
  for (int i = n_rad - 1; i >= 0; --i) {
    const cplx* uc = Uc + (size_t)i * (W + 1);
    const cplx t = cadd(p.y[(size_t)i * ld + a], pw[0]);
    const cplx xi = cmul(t, uc[0]);
    p.y[(size_t)i * ld + a] = xi;
    // Ucol[.][1] is pre-scaled by 1/U[i][i]: it multiplies (y_i + pw0), not x_i
    if (W >= 1) { pw[0] = pw[1]; cfms(pw[0], uc[1], t); }
    for (int d = 1; d < W; ++d) { pw[d] = pw[d + 1]; cfms(pw[d], uc[d + 1], xi); }
  }
}

template <int W>
static int launch_precond_w(const PrecArgs& a, cudaStream_t s) {
  const size_t smem = PrecPlan<W>::smem(a.tile_rows);
  if (cudaFuncSetAttribute(k_precond_tile<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
  int n = 0;
  if (a.P > 1) {
    if (!a.spikes_done) {
      const size_t ssmem = (size_t)2 * TDDE_AP_MAXC * SPK_ROWS * 2 * W * sizeof(cplx);
      if (cudaFuncSetAttribute(k_precond_spikes<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ssmem) != cudaSuccess) return -2;
      k_precond_spikes<W><<<dim3((a.ld + 127) / 128, a.P), 128, ssmem, s>>>(a);
      ++n;
    }
    k_precond_schur<W><<<a.ld / PC_NT, PC_NT * W, 0, s>>>(a);
    k_precond_corners<W><<<dim3((a.ld + 127) / 128, a.P - 1), 128, 0, s>>>(a);
    n += 2;
  }
  k_precond_tile<W><<<dim3(a.ld / PC_NT, a.P), PC_NT, smem, s>>>(a);
  return n + 1;
}

template <int W>
static int launch_vec_spikes_w(const VecArgs& v, const PrecArgs& a, int mode, cudaStream_t s) {
  const size_t smem = (size_t)2 * TDDE_AP_MAXC * VSP_ROWS * 2 * W * sizeof(cplx);
  dim3 grid((a.ld + 127) / 128, a.P);
  if (mode == 0) {
    if (cudaFuncSetAttribute(k_vec_spikes<W, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
    k_vec_spikes<W, 0><<<grid, 128, smem, s>>>(v, a);
  } else {
    if (cudaFuncSetAttribute(k_vec_spikes<W, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
    k_vec_spikes<W, 1><<<grid, 128, smem, s>>>(v, a);
  }
  return 1;
}

// the p-update (mode 0) or the s-update (mode 1) fused with the spike products of the vector it writes; -1: not available
// for this problem (no partitions, or an untemplated bandwidth): the caller runs the plain update and the full solve
int launch_vec_spikes(const VecArgs& v, const PrecArgs& a, int mode, cudaStream_t s) {
  if (a.P <= 1 || (long long)((a.ld + 127) / 128) * a.P > TDDE_MAX_PARTIAL_BLOCKS) return -1;
  switch (a.w) {
#define X(W) case W: return launch_vec_spikes_w<W>(v, a, mode, s);
    TDDE_PC_WIDTHS(X)
#undef X
    default: return -1;
  }
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
