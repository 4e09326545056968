// tdde_apply_sparse.cu -- operator apply for general sparse angular couplings A_L (Eq. 17;
// selection-rule-sparse H^theta: PAPER.md:231-245).
//
//   y[a', i] = sum_j Blk_{k(a')}[i, j] x[a', j]  +  beta * sum_L g_L sum_a A_L[a', a] sum_j R_L[i, j] x[a, j]
//
// Same organisation as the banded register-A kernel (tdde_apply.cu): lane <-> channel a', a thread walks a radial segment in
// scatter form with the 2W+1 pending outputs in a register window; the x tile (the CTA's 128 channels plus every channel they
// couple to), the radial column coefficients of all terms and the block coefficients of the CTA's kappa-classes arrive by 1-D
// TMA bulk copies in a two-stage mbarrier ring.  What differs: A_L is an arbitrary sparse matrix, any number of terms up to
// TDDE_MAX_TERMS, per-term bandwidths up to W.  The rows of A_L (ELL: values pre-multiplied by beta g_L, column positions
// absolute channel index) live in SHARED memory, one column per thread, loaded once per CTA, when they fit, and are otherwise read
// from global memory (L1/L2) once per input row; the angular combination
// z_L = sum_q A_L[a', q] x[col_q] is formed per input row and pushed through the radial band from warp-broadcast coefficients.
#include "tdde_reduce.cuh"

#define SP_NC TDDE_AP_NC
#define SP_JC 4
#define SP_NST 2
#define SP_MAXC TDDE_AP_MAXC

namespace {
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok)
                 : "r"(smem_u32(bar)), "r"(parity)
                 : "memory");
  } while (!ok);
}
}  // namespace

// complex elements of one pipeline stage
__host__ __device__ inline size_t sparse_stage_elems(int W, int T, int xw) {
  const int ND = 2 * W + 1;
  return (size_t)SP_JC * T * ND + (size_t)SP_MAXC * SP_JC * ND + (size_t)SP_JC * xw;
}
size_t apply_sparse_smem(int W, int T, int nslots, int xw, bool a_in_smem) {
  return (a_in_smem ? (size_t)nslots * SP_NC * (sizeof(cplx) + sizeof(int)) : 0) + SP_NST * sparse_stage_elems(W, T, xw) * sizeof(cplx) +
         TDDE_MAX_TERMS * sizeof(cplx) + 64;
}

template <int W>
__global__ void __launch_bounds__(SP_NC, 1) k_apply_sparse(const __grid_constant__ ApplyArgs p) {
  constexpr int ND = 2 * W + 1, JC = SP_JC;
  if (p.guard == 1 && solver_idle(p.red.st)) return;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int T = p.n_terms, S = p.sp_nslots, XW = p.sp_xw;
  const size_t stage = sparse_stage_elems(W, T, XW);
  const int RS = JC * T * ND, BS = SP_MAXC * JC * ND;
  cplx* stage_base = reinterpret_cast<cplx*>(smem_raw);
  cplx* coefL = stage_base + SP_NST * stage;                 // [TDDE_MAX_TERMS] beta g_L
  cplx* Av_s = coefL + TDDE_MAX_TERMS;                       // [S][128] (only when sp_a_smem)
  const size_t Sa = p.sp_a_smem ? (size_t)S : 0;
  int* Ac_s = reinterpret_cast<int*>(Av_s + Sa * SP_NC);     // [S][128]
  uint64_t* full = reinterpret_cast<uint64_t*>(Ac_s + Sa * SP_NC);               // S * 128 ints: 8-byte aligned

  const int tid = threadIdx.x, ld = p.ld, n_rad = p.n_rad;
  const int a0 = blockIdx.x * SP_NC, a = a0 + tid;
  const bool lane_ok = a >= p.own_lo && a < p.own_hi;          // own_hi <= ld
  const int ac = a < ld ? a : ld - 1;
  const int i0 = blockIdx.y * p.seg_len, i1 = min(n_rad, i0 + p.seg_len);
  const int jlo = max(0, i0 - W), jhi = min(n_rad, i1 + W), jend = i1 + W;
  const int nchunks = (jend - jlo + JC - 1) / JC;
  const int slot = p.slot[ac];
  const cplx* blk_g = p.blk + (size_t)p.cls[ac] * n_rad * ND;

  // x tile: columns [win_lo, win_lo + XW) of a row; either the whole row or the CTA's channels plus the coupling reach on each side
  const int win_lo = p.sp_full ? 0 : a0 - p.sp_reach;
  const int xa_lo = max(0, win_lo), xa_hi = min(ld, win_lo + XW);
  const int x_dst_off = xa_lo - win_lo;
  const uint32_t x_bytes = (uint32_t)(xa_hi - xa_lo) * sizeof(cplx);
  const int* cta_cls = p.cta_cls + blockIdx.x * SP_MAXC;

  for (size_t q = tid; q < SP_NST * stage; q += SP_NC) stage_base[q] = make_double2(0, 0);
  // rows of A_L for this thread's channel: copied to shared memory when they fit (own column of the shared arrays: no hazard),
  // otherwise read from global memory per row; the factor beta g_L is applied to z_L
  if (tid < T) {
    const double* g = p.g + (p.step_ptr ? (size_t)(*p.step_ptr) * T : 0);
    coefL[tid] = make_double2(p.beta.x * g[tid], p.beta.y * g[tid]);
  }
  if (p.sp_a_smem) {
    for (int s = 0; s < S; ++s) {
      Av_s[(size_t)s * SP_NC + tid] = p.sp_val[(size_t)s * ld + ac];
      Ac_s[(size_t)s * SP_NC + tid] = p.sp_col[(size_t)s * ld + ac];
    }
  }
  const cplx* Av = p.sp_a_smem ? Av_s + tid : p.sp_val + ac;
  const int* Ac = p.sp_a_smem ? Ac_s + tid : p.sp_col + ac;
  const size_t astr = p.sp_a_smem ? SP_NC : ld;
  if (tid == 0) {
    for (int q = 0; q < SP_NST; ++q) mbar_init(&full[q], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");

  auto issue = [&](int c) {                                  // one elected thread: all bulk copies of chunk c
    cplx* st = stage_base + (size_t)(c % SP_NST) * stage;
    uint64_t* bar = &full[c % SP_NST];
    const int j = jlo + c * JC;
    const int nr = min(JC, jhi - j);
    if (nr <= 0) return;
    int ncls = 0;
#pragma unroll
    for (int q = 0; q < SP_MAXC; ++q) ncls += (cta_cls[q] >= 0);
    uint32_t bytes = (uint32_t)nr * x_bytes + (uint32_t)ncls * nr * ND * sizeof(cplx) + (uint32_t)nr * T * ND * sizeof(cplx);
    mbar_expect_tx(bar, bytes);
    if (T > 0) bulk_g2s(st, p.Rall + (size_t)j * T * ND, (uint32_t)nr * T * ND * sizeof(cplx), bar);
#pragma unroll
    for (int q = 0; q < SP_MAXC; ++q) {
      const int kk = cta_cls[q];
      if (kk >= 0) bulk_g2s(st + RS + (size_t)q * JC * ND, p.blk + ((size_t)kk * n_rad + j) * ND, (uint32_t)nr * ND * sizeof(cplx), bar);
    }
    for (int r = 0; r < nr; ++r)
      bulk_g2s(st + RS + BS + (size_t)r * XW + x_dst_off, p.x + (size_t)(j + r) * ld + xa_lo, x_bytes, bar);
  };
  if (tid == 0) {
    for (int c = 0; c < SP_NST && c < nchunks; ++c) issue(c);
  }

  cplx yw[ND];
#pragma unroll
  for (int e = 0; e < ND; ++e) yw[e] = make_double2(0, 0);
  cplx d0 = make_double2(0, 0);
  double d1 = 0;
  const int own = a - win_lo;                                // this thread's own column in the x tile (lanes beyond ld read zeros)
  for (int c = 0; c < nchunks; ++c) {
    const cplx* st = stage_base + (size_t)(c % SP_NST) * stage;
    const int jc0 = jlo + c * JC;
    const int nr_real = min(JC, jhi - jc0), nr_all = min(JC, jend - jc0);
    if (nr_real > 0) mbar_wait(&full[c % SP_NST], (c / SP_NST) & 1);
    for (int r = 0; r < nr_all; ++r) {
      const int i = jc0 + r - W;                             // the output row completed by input row jc0 + r
      const bool emit = (i >= i0) && lane_ok;
      if (r < nr_real) {
        const cplx* xs = st + RS + BS + (size_t)r * XW;
        const cplx x0 = lane_ok ? xs[own] : make_double2(0, 0);
        if (slot >= 0) {
          const cplx* bc = st + RS + ((size_t)slot * JC + r) * ND;
#pragma unroll
          for (int e = 0; e < ND; ++e) cfma(yw[e], bc[e], x0);
        } else {
          const cplx* bc = blk_g + (size_t)(jc0 + r) * ND;
#pragma unroll
          for (int e = 0; e < ND; ++e) cfma(yw[e], __ldg(bc + e), x0);
        }
        int s = 0;
        const cplx* xw0 = xs - win_lo;                        // absolute channel index -> tile column
#pragma unroll 1
        for (int L = 0; L < T; ++L) {
          cplx z0 = make_double2(0, 0), z1 = make_double2(0, 0);
          const int ns = p.sp_nslot[L];
          int q = 0;
          constexpr int U = W >= 13 ? 4 : 8;                  // loads in flight per thread (the rows of A_L may come from L2)
          for (; q + U <= ns; q += U, s += U) {
            cplx av[U];
            int ci[U];
#pragma unroll
            for (int u = 0; u < U; ++u) { av[u] = Av[(size_t)(s + u) * astr]; ci[u] = Ac[(size_t)(s + u) * astr]; }
#pragma unroll
            for (int u = 0; u < U; u += 2) { cfma(z0, av[u], xw0[ci[u]]); cfma(z1, av[u + 1], xw0[ci[u + 1]]); }
          }
          for (; q < ns; ++q, ++s) cfma(z0, Av[(size_t)s * astr], xw0[Ac[(size_t)s * astr]]);
          const cplx z = cmul(coefL[L], cadd(z0, z1));
          const cplx* rc = st + ((size_t)r * T + L) * ND;    // warp-uniform: broadcast LDS.128
#pragma unroll
          for (int e = 0; e < ND; ++e) cfma(yw[e], rc[e], z);
        }
      }
      if (emit) {
        cplx yv = yw[0];
        const cplx ax = p.aux ? p.aux[(size_t)i * ld + a] : make_double2(0, 0);
        if (p.emode == 2) {                                  // ||b||^2 = ||S c + r0 / 2||^2, nothing stored
          yv.x = fma(0.5, ax.x, yv.x); yv.y = fma(0.5, ax.y, yv.y);
        } else {
          if (p.emode == 1) { yv = cmul(p.oscale, yv); p.y2[(size_t)i * ld + a] = yv; }
          p.y[(size_t)i * ld + a] = yv;
          cfma_conj(d0, ax, yv);
        }
        d1 = fma(yv.x, yv.x, d1); d1 = fma(yv.y, yv.y, d1);
      }
#pragma unroll
      for (int e = 0; e < ND - 1; ++e) yw[e] = yw[e + 1];
      yw[ND - 1] = make_double2(0, 0);
    }
    __syncthreads();                                         // everybody is done with stage c % SP_NST
    if (tid == 0 && c + SP_NST < nchunks) issue(c + SP_NST);
  }
  if (p.red.fin != FIN_NONE) grid_reduce_finalize<SP_NC>(d0.x, d0.y, d1, p.red);
}

int launch_apply_sparse(const ApplyArgs& a, int W, cudaStream_t s) {
  dim3 grid((a.ld + SP_NC - 1) / SP_NC, (a.n_rad + a.seg_len - 1) / a.seg_len);
  const size_t smem = apply_sparse_smem(W, a.n_terms, a.sp_nslots, a.sp_xw, a.sp_a_smem != 0);
#define X(w)                                                                                                           \
  if (W == w) {                                                                                                        \
    if (cudaFuncSetAttribute(k_apply_sparse<w>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2; \
    k_apply_sparse<w><<<grid, SP_NC, smem, s>>>(a);                                                                    \
    return 1;                                                                                                          \
  }
  X(3) X(6) X(9) X(13)
#undef X
  return -1;
}
