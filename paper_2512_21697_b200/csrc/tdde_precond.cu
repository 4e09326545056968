// tdde_precond.cu -- y = (S + i dt/2 H0)^{-1} x as batched banded triangular solves (
// PAPER.md:211-215, Eq. 26: M is block-diagonal over angular channels, LU factors computed at start-up).
//
// One warp per 32 consecutive angular channels, lane = channel (coalesced 16-byte accesses in the internal
// layout); the recurrence along r is inherently serial, so the kernel is organised around two facts:
//  * latency of the dependent chain.  Both sweeps run in column-oriented (axpy) form: once y_i is final the W
//    pending rows below it are updated independently.  Only the update of the next row is on the critical
//    path, and it is split as  pw0' = (pw1 - c x_i) - c pw0  so that the chain is one complex FMA (two
//    dependent DFMAs) per row; for the U sweep the host pre-scales U[i-1][i] by 1/U[i][i] for the same reason.
//  * few warps (N_ang / 32), so memory latency cannot be hidden by occupancy.  Vector rows and the factor rows
//    of the (few) kappa-classes present in the warp are streamed through a shared-memory ring with cp.async,
//    PC_STAGES x PC_ROWS rows ahead of the row being solved.
// Factor layout (tdde_create.cu): Lcol[k][i][d-1] = L[i+d][i];
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
  static constexpr size_t SMEM = (size_t)PC_STAGES * STAGE * sizeof(cplx);
};

// Kernel A of the partitioned solve (and the whole solve when P == 1): one warp = 32 channels x one row range.
// Factor rows of the warp's kappa-classes stream through a cp.async ring in shared memory; the vector rows of the
// next stage are prefetched into registers while the current stage is being solved.
template <int W>
__global__ void __launch_bounds__(PC_NT) k_precond(const PrecArgs p) {
  using PL = PrecPlan<W>;
  if (p.st && solver_idle(p.st)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* ring = reinterpret_cast<cplx*>(smem_raw);
  const int lane = threadIdx.x;
  const int a = blockIdx.x * PC_NT + lane;                           // a < ld always (ld is a multiple of 32)
  const int ld = p.ld, n_tot = p.n_rad;
  // rows [row0, row0 + n_rad): interior blockIdx.y plus the separator after it (identity rows in the factors)
  const int row0 = p.range_lo[blockIdx.y];
  const int n_rad = p.range_lo[blockIdx.y + 1] - row0;
  const cplx* xin = p.x + (size_t)row0 * ld + a;
  cplx* yout = p.y + (size_t)row0 * ld + a;
  const int* wcls = p.warp_cls + blockIdx.x * PC_MAXC;
  int ncls = 0;
#pragma unroll
  for (int q = 0; q < PC_MAXC; ++q) ncls += (wcls[q] >= 0);
  const int slot = p.slot[a];
  const int k = p.cls[a];
  const int nst = (n_rad + PC_ROWS - 1) / PC_ROWS;

  cplx pw[W + 1];
  cplx xn[PC_ROWS];

  // ================= forward: L y = x =================
  {
    auto issue = [&](int s) {                                        // factor rows [s*R, s*R + R) of every class
      if (s < nst) {
        cplx* st = ring + (size_t)(s % PC_STAGES) * PL::STAGE;
        const int r0 = s * PC_ROWS, nr = min(PC_ROWS, n_rad - r0);
        for (int q = 0; q < ncls; ++q) {
          const cplx* src = p.Lcol + ((size_t)wcls[q] * n_tot + row0 + r0) * W;
          cplx* dst = st + (size_t)q * PC_ROWS * PL::CW;
          for (int e = lane; e < nr * W; e += PC_NT) cp_async16(dst + e, src + e);
        }
      }
      cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
    for (int s = 0; s < PC_STAGES - 1; ++s) issue(s);
#pragma unroll
    for (int r = 0; r < PC_ROWS; ++r) xn[r] = xin[(size_t)min(r, n_rad - 1) * ld];
    for (int s = 0; s < nst; ++s) {
      const int r0 = s * PC_ROWS, nr = min(PC_ROWS, n_rad - r0);
      cplx xc[PC_ROWS];
#pragma unroll
      for (int r = 0; r < PC_ROWS; ++r) xc[r] = xn[r];
      if (r0 + 2 * PC_ROWS <= n_rad) {                               // next stage is full: no clamping
        const cplx* xp = xin + (size_t)(r0 + PC_ROWS) * ld;
#pragma unroll
        for (int r = 0; r < PC_ROWS; ++r) { xn[r] = *xp; xp += ld; }
      } else if (s + 1 < nst) {
#pragma unroll
        for (int r = 0; r < PC_ROWS; ++r) xn[r] = xin[(size_t)min(r0 + PC_ROWS + r, n_rad - 1) * ld];
      }
      issue(s + PC_STAGES - 1);
      cp_async_wait<PC_STAGES - 1>();
      __syncwarp();
      const cplx* cs = ring + (size_t)(s % PC_STAGES) * PL::STAGE + (size_t)(slot >= 0 ? slot : 0) * PC_ROWS * PL::CW;
      const cplx* cg = p.Lcol + ((size_t)k * n_tot + row0 + r0) * W;
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
          yout[(size_t)(r0 + r) * ld] = yi;
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
        for (int q = 0; q < ncls; ++q) {
          const cplx* src = p.Ucol + ((size_t)wcls[q] * n_tot + row0 + lo) * (W + 1);
          cplx* dst = st + (size_t)q * PC_ROWS * PL::CW;
          for (int e = lane; e < nr * (W + 1); e += PC_NT) cp_async16(dst + e, src + e);
        }
      }
      cp_async_commit();
    };
#pragma unroll
    for (int d = 0; d <= W; ++d) pw[d] = make_double2(0, 0);
    for (int s = 0; s < PC_STAGES - 1; ++s) issue(s);
    // xn[r] holds row (hi - 1 - r) of the stage: the order in which the sweep consumes them
#pragma unroll
    for (int r = 0; r < PC_ROWS; ++r) xn[r] = yout[(size_t)max(n_rad - 1 - r, 0) * ld];
    for (int s = 0; s < nst; ++s) {
      const int hi = n_rad - s * PC_ROWS, lo = max(0, hi - PC_ROWS), nr = hi - lo;
      cplx xc[PC_ROWS];
#pragma unroll
      for (int r = 0; r < PC_ROWS; ++r) xc[r] = xn[r];
      if (lo >= PC_ROWS) {                                           // next stage is full: no clamping
        const cplx* xp = yout + (size_t)(lo - 1) * ld;
#pragma unroll
        for (int r = 0; r < PC_ROWS; ++r) { xn[r] = *xp; xp -= ld; }
      } else if (s + 1 < nst) {
#pragma unroll
        for (int r = 0; r < PC_ROWS; ++r) xn[r] = yout[(size_t)max(lo - 1 - r, 0) * ld];
      }
      issue(s + PC_STAGES - 1);
      cp_async_wait<PC_STAGES - 1>();
      __syncwarp();
      const cplx* cs = ring + (size_t)(s % PC_STAGES) * PL::STAGE + (size_t)(slot >= 0 ? slot : 0) * PC_ROWS * PL::CW;
      const cplx* cg = p.Ucol + ((size_t)k * n_tot + row0 + lo) * (W + 1);
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

// ---- kernel B: Schur-complement solve for the separator unknowns (tdde_partition.h), two fully parallel steps ----
// B1: r_S = b_S - A_SI t_I from the separator rows of M: one thread per (separator row, channel).
template <int W>
__global__ void __launch_bounds__(128) k_precond_schur_rhs(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * 128 + threadIdx.x;
  if (a >= p.ld) return;
  constexpr int ND = 2 * W + 1;
  const int srow = blockIdx.y, ld = p.ld, n_rad = p.n_rad;
  const int i = p.int_hi[srow / W] + srow % W;
  const cplx* ms = p.Msep + ((size_t)p.cls[a] * p.ns + srow) * ND;
  cplx acc = p.y[(size_t)i * ld + a];
#pragma unroll
  for (int d = -W; d <= W; ++d) {
    const int ii = i + d;
    if (ii >= 0 && ii < n_rad) {
      const cplx m = __ldg(ms + d + W);
      cfma(acc, make_double2(-m.x, -m.y), p.y[(size_t)ii * ld + a]);
    }
  }
  p.rs[(size_t)srow * ld + a] = acc;
}
// B2: x_S = Sc^{-1} r_S (dense (P-1) w square per class): one thread per (separator row, channel).
template <int W>
__global__ void __launch_bounds__(128) k_precond_schur_mul(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  const int a = blockIdx.x * 128 + threadIdx.x;
  if (a >= p.ld) return;
  const int o = blockIdx.y, ld = p.ld, ns = p.ns;
  const cplx* sc = p.Scinv + ((size_t)p.cls[a] * ns + o) * ns;
  cplx acc[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) acc[u] = make_double2(0, 0);
  int q = 0;
  for (; q + 3 < ns; q += 4) {
#pragma unroll
    for (int u = 0; u < 4; ++u) cfma(acc[u], __ldg(sc + q + u), p.rs[(size_t)(q + u) * ld + a]);
  }
  for (; q < ns; ++q) cfma(acc[0], __ldg(sc + q), p.rs[(size_t)q * ld + a]);
  const int row = p.int_hi[o / W] + o % W;
  p.y[(size_t)row * ld + a] = cadd(cadd(acc[0], acc[1]), cadd(acc[2], acc[3]));
}

// ---- kernel C: x_I = t_I - E^- x_S(before) - E^+ x_S(after): streaming, 2 W complex FMAs per row ----
// CTA = 128 channels x PCC_ROWS interior rows.  The spike rows of the CTA's kappa-classes (same class list as the
// operator apply) are staged in shared memory with cp.async and read back as warp-broadcasts; each thread first
// issues all of its vector loads, so enough bytes are in flight to stream at HBM speed.
#ifndef PCC_ROWS
#define PCC_ROWS 8
#endif
template <int W>
__global__ void __launch_bounds__(128) k_precond_correct(const PrecArgs p) {
  if (p.st && solver_idle(p.st)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* Es = reinterpret_cast<cplx*>(smem_raw);                     // [TDDE_AP_MAXC][PCC_ROWS][2W]
  const int q = blockIdx.y, ld = p.ld;
  const int lo = p.range_lo[q], hi = p.int_hi[q];
  const int i0 = lo + blockIdx.z * PCC_ROWS;
  if (i0 >= hi) return;
  const int nr = min(PCC_ROWS, hi - i0);
  const int a = blockIdx.x * 128 + threadIdx.x;
  const bool ok = a < ld;
  const int ac = ok ? a : ld - 1;
  const int* ccls = p.cta_cls + blockIdx.x * TDDE_AP_MAXC;
  for (int s = 0; s < TDDE_AP_MAXC; ++s) {
    const int k = ccls[s];
    if (k < 0) break;
    const cplx* src = p.Esp + ((size_t)k * p.n_rad + i0) * 2 * W;
    cplx* dst = Es + (size_t)s * PCC_ROWS * 2 * W;
    for (int e = threadIdx.x; e < nr * 2 * W; e += 128) cp_async16(dst + e, src + e);
  }
  cp_async_commit();
  cplx t[PCC_ROWS];
#pragma unroll
  for (int r = 0; r < PCC_ROWS; ++r) t[r] = (r < nr) ? p.y[(size_t)(i0 + r) * ld + ac] : make_double2(0, 0);
  cplx xm[W], xp[W];
#pragma unroll
  for (int c = 0; c < W; ++c) {
    xm[c] = q > 0 ? p.y[(size_t)(p.int_hi[q - 1] + c) * ld + ac] : make_double2(0, 0);
    xp[c] = q + 1 < p.P ? p.y[(size_t)(hi + c) * ld + ac] : make_double2(0, 0);
    xm[c] = make_double2(-xm[c].x, -xm[c].y);
    xp[c] = make_double2(-xp[c].x, -xp[c].y);
  }
  cp_async_wait<0>();
  __syncthreads();
  const int slot = p.aslot[ac];
  const cplx* Eg = p.Esp + ((size_t)p.cls[ac] * p.n_rad + i0) * 2 * W;
  const cplx* El = Es + (size_t)(slot >= 0 ? slot : 0) * PCC_ROWS * 2 * W;
#pragma unroll
  for (int r = 0; r < PCC_ROWS; ++r) {
    if (r < nr) {
      cplx v = t[r];
      if (slot >= 0) {
#pragma unroll
        for (int c = 0; c < W; ++c) { cfma(v, El[r * 2 * W + c], xm[c]); cfma(v, El[r * 2 * W + W + c], xp[c]); }
      } else {
#pragma unroll
        for (int c = 0; c < W; ++c) { cfma(v, __ldg(Eg + r * 2 * W + c), xm[c]); cfma(v, __ldg(Eg + r * 2 * W + W + c), xp[c]); }
      }
      if (ok) p.y[(size_t)(i0 + r) * ld + a] = v;
    }
  }
}

// runtime-w fallback (w <= 32): pending rows in a small local array, direct global loads
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
  static bool attr_set = false;
  const size_t smem = PrecPlan<W>::SMEM;
  const size_t csmem = (size_t)TDDE_AP_MAXC * PCC_ROWS * 2 * W * sizeof(cplx);
  static_assert(TDDE_AP_NC == 128, "k_precond_correct shares the apply's 128-channel class lists");
  if (!attr_set) {
    if (cudaFuncSetAttribute(k_precond<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
    if (cudaFuncSetAttribute(k_precond_correct<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)csmem) != cudaSuccess) return -2;
    attr_set = true;
  }
  k_precond<W><<<dim3(a.ld / PC_NT, a.P), PC_NT, smem, s>>>(a);
  if (a.P == 1) return 1;
  k_precond_schur_rhs<W><<<dim3((a.ld + 127) / 128, a.ns), 128, 0, s>>>(a);
  k_precond_schur_mul<W><<<dim3((a.ld + 127) / 128, a.ns), 128, 0, s>>>(a);
  int max_int = 0;
  for (int q = 0; q < a.P; ++q) max_int = max_int > a.int_hi[q] - a.range_lo[q] ? max_int : a.int_hi[q] - a.range_lo[q];
  k_precond_correct<W><<<dim3((a.ld + 127) / 128, a.P, (max_int + PCC_ROWS - 1) / PCC_ROWS), 128, csmem, s>>>(a);
  return 4;
}

int launch_precond(const PrecArgs& a, cudaStream_t s) {
  switch (a.w) {
    case 3: return launch_precond_w<3>(a, s);
    case 6: return launch_precond_w<6>(a, s);
    case 9: return launch_precond_w<9>(a, s);
    case 13: return launch_precond_w<13>(a, s);
    default:
      if (a.w > 32 || a.w < 1 || a.P != 1) return -1;
      k_precond_any<<<(a.ld + PC_NT - 1) / PC_NT, PC_NT, 0, s>>>(a);
  }
  return 1;
}
