// tdde_apply.cu -- structure-aware, matrix-free operator apply (Eq. 17)
//
//   y[a', i] = sum_j Blk_{k(a')}[i, j] x[a', j]  +  beta * sum_L g_L sum_a A_L[a', a] sum_j R_L[i, j] x[a, j]
//
// The assembled matrix is never formed.  Per term the cheaper factorisation is used: first the angular
// combination z_L[a', j] = sum_a A_L[a', a] x[a, j]  (nnz_row(A_L) complex FMAs), then the radial band
// y[a', i] += R_L[i, j] z_L[a', j]  (2w+1 complex FMAs), i.e. n_d + sum_L (n_d + nnz_row(A_L)) cFMA per element.
//
// Banded fast path (A_L non-zero only at channel offsets 1 <= |o| <= m_L, m_L = M0 + MS * L):
//   lane <-> channel a', a thread walks a radial segment in scatter ("column") form.
//   * A_L[a', a'+o] * beta * g_L are loaded once into registers (the angular coupling is applied from registers);
//   * x[j, a'+o] are coalesced 16-byte loads shared by every term that has the offset o;
//   * R_L[:, j] column coefficients are warp-uniform (one address per warp);
//   * the 2W+1 pending outputs y[j-W .. j+W] are a register window; when row j has been consumed output
//     j-W is complete, is written once (coalesced) and enters the fused inner products.
// This kernel is FP64-FMA bound (27-52 flop per HBM byte), not HBM bound.
#include <algorithm>
#include "tdde_reduce.cuh"

#define AP_NT 128            // generic kernel: threads per block
#define AP_MINB TDDE_AP_MINB
#define AP_NC TDDE_AP_NC      // banded kernel: channels per CTA
#define AP_JC TDDE_AP_JC      // radial rows per pipeline stage
#define AP_MAXC TDDE_AP_MAXC  // distinct kappa-classes per CTA staged in shared memory

template <int T, int M0, int MS>
struct BandShape {
  __host__ __device__ static constexpr int m(int L) { return M0 + MS * L; }
  __host__ __device__ static constexpr int maxm() { return T == 0 ? 0 : M0 + MS * (T - 1); }
  __host__ __device__ static constexpr int slot0(int L) {           // first slot of term L; slots per term = 2 m_L
    int s = 0;
    for (int l = 0; l < L; ++l) s += 2 * m(l);
    return s;
  }
  __host__ __device__ static constexpr int nslots() { return slot0(T); }
};

// ---- TMA (1-D bulk async copy) + mbarrier helpers: raw PTX, sm_90+ ----
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
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
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

// Shared-memory plan of one pipeline stage (JC radial rows):
//   Rs[JC][T][ND]     radial column coefficients of every term (one bulk copy: host stores them [n_rad][T][ND])
//   Bs[MAXC][JC][ND]  block column coefficients of the (at most MAXC) distinct kappa-classes of this CTA
//   Xs[JC][XW]        x rows of the CTA's 128 channels plus MAXM halo channels on each side (one bulk copy per row)
// plus Ps[2][JC][128]: partial outputs handed from warp group 1 to warp group 0 (double-buffered).
template <int T, int M0, int MS, int W, int NG, bool BLK>
struct ApplyPlan {
  using SH = BandShape<T, M0, MS>;
  static constexpr int ND = 2 * W + 1;
  static constexpr int MAXM = SH::maxm();
  static constexpr int XW = AP_NC + 2 * MAXM;
  // rows per stage: the two-group variant (one CTA per SM) takes twice as many when the shared memory allows,
  // which halves the number of CTA barriers (measured: HBM-scale 2.41 -> 2.25 ms)
  // BLK == false (in-iteration applies): the fused-dot operand and the vector replacing the block part reach the row loop
  // through a per-thread cp.async double buffer instead of plain global loads inside it
  static constexpr bool VST = !BLK && T > 0;
  // W >= 9: the 2W+1-entry window and all A_L registers do not fit 255 registers.  Each warp group keeps the row of its widest
  // term in shared memory instead (one column per thread, conflict-free 16-byte loads) -- no spills.
  static constexpr bool ASM = W >= 9 && T > 0;
  static constexpr int AS = ASM ? NG * 2 * MAXM * AP_NC : 0;
  __host__ __device__ static constexpr size_t smem_for(int jc) {
    return (size_t)(3 * (jc * T * ND + (BLK ? AP_MAXC * jc * ND : 0) + jc * XW) + ((T > 0 && NG == 2) ? 2 * jc * AP_NC : 0) +
                    (VST ? 4 * jc * AP_NC : 0) + AS) * sizeof(cplx) + 64;
  }
  static constexpr int JC = (NG == 2 && smem_for(2 * AP_JC) <= 220 * 1024) ? 2 * AP_JC : AP_JC;
  static constexpr int RS = JC * T * ND;                    // complex elements
  static constexpr int BS = BLK ? AP_MAXC * JC * ND : 0;   // no block part: no class coefficients staged
  static constexpr int XS = JC * XW;
  static constexpr int STAGE = RS + BS + XS;
  static constexpr int PS = (T > 0 && NG == 2) ? 2 * JC * AP_NC : 0;
  static constexpr int VS = VST ? 4 * JC * AP_NC : 0;       // [2 buffers][aux, addv][JC][AP_NC]
  static constexpr int NSTAGE = 3;
  static constexpr size_t SMEM = (size_t)(NSTAGE * STAGE + PS + VS + AS) * sizeof(cplx) + 64;
  // Term split: the terms of one channel are shared between two warp groups so that each thread keeps only about
  // half of the A_L registers (4 warps per SM sub-partition instead of 2).  Group 0 also owns the block part, the
  // write-out and the fused inner products.  Greedy balance of complex FMAs per row, largest term first.
  __host__ __device__ static constexpr int cost(int L) { return ND + 2 * SH::m(L); }
  __host__ __device__ static constexpr int mask() {          // bit L set: term L belongs to group 1
    int c0 = (BLK ? ND : 0) + 4, c1 = 0, mk = 0;
    for (int L = T - 1; L >= 0; --L) {
      if (c1 < c0) { c1 += cost(L); mk |= 1 << L; } else c0 += cost(L);
    }
    return mk;
  }
  __host__ __device__ static constexpr bool mine(int G, int L) { return NG == 1 || ((mask() >> L) & 1) == G; }
  __host__ __device__ static constexpr int wide(int G) {     // the group's widest term (its A_L row lives in shared memory when ASM)
    int best = -1;
    for (int L = 0; L < T; ++L) if (mine(G, L) && (best < 0 || SH::m(L) > SH::m(best))) best = L;
    return best;
  }
  __host__ __device__ static constexpr int gmaxm(int G) {    // largest channel offset the group touches
    int m = 0;
    for (int L = 0; L < T; ++L) if (mine(G, L) && SH::m(L) > m) m = SH::m(L);
    return m;
  }
};

struct ApplyCommon {
  int tid, a, ac, ld, n_rad, i0, i1, jlo, jhi, jend, nchunks, slot;
  bool lane_ok;
  cplx* stage_base;
  cplx* Ps;
  cplx* Vs;
  cplx* As;             // ASM: [NG][2 MAXM][AP_NC] row of each group's widest term
  uint64_t* full;       // [NSTAGE] TMA landed
  uint64_t* pfull;      // [2] group 1 has published its partial rows of a chunk
  uint64_t* pempty;     // [2] group 0 has consumed them
  const cplx* blk_g;
};

// Work of one warp group G over the whole radial segment (see k_apply_banded).
template <int T, int M0, int MS, int W, int NG, bool BLK, int G, class IssueFn>
__device__ __forceinline__ void apply_group(const ApplyArgs& p, const ApplyCommon& k, IssueFn issue, cplx& d0, double& d1) {
  using SH = BandShape<T, M0, MS>;
  using PL = ApplyPlan<T, M0, MS, W, NG, BLK>;
  constexpr int ND = PL::ND, MAXM = PL::MAXM, NS = SH::nslots(), XW = PL::XW, JC = PL::JC, GM = PL::gmaxm(G);
  constexpr bool SPLIT = (NG == 2) && (T > 0);
  constexpr int RU = (W >= 9 && T > 0) ? TDDE_AP_RU9 : ((T == 0) ? 4 : TDDE_AP_RU);   // rows unrolled together (register pressure vs ILP)
  const int ld = k.ld;

  // angular coefficients of this group's terms in registers, pre-multiplied by beta * g_L
  cplx Areg[NS > 0 ? NS : 1];
  constexpr int LW = PL::ASM ? PL::wide(G) : -1;
  cplx* const As = k.As + (size_t)G * 2 * MAXM * AP_NC + k.tid;   // this thread's column
  if (T > 0) {
    const double* g = p.g + (p.step_ptr ? (size_t)(*p.step_ptr) * T : 0);
#pragma unroll
    for (int L = 0; L < T; ++L) {
      if (!PL::mine(G, L)) continue;
      const double gl = g[L];
      const cplx coef = make_double2(p.beta.x * gl, p.beta.y * gl);
#pragma unroll
      for (int q = 0; q < 2 * SH::m(L); ++q) {
        const int s = SH::slot0(L) + q;
        if (L == LW) As[q * AP_NC] = cmul(coef, p.Aoff[(size_t)s * ld + k.ac]);
        else Areg[s] = cmul(coef, p.Aoff[(size_t)s * ld + k.ac]);
      }
    }
  }
  cplx yw[ND];
#pragma unroll
  for (int e = 0; e < ND; ++e) yw[e] = make_double2(0, 0);

  // Group 1 runs ahead: it publishes its partial rows of chunk c in Ps[c & 1] and signals pfull[c & 1]; group 0 waits for that,
  // finishes every output row of the chunk (sum, store, fused inner products) and signals pempty[c & 1].  Nobody waits at a
  // CTA-wide barrier: group 1 only blocks when it is two chunks ahead, group 0 only on group 1's chunk.  A stage buffer is
  // refilled (chunk c + 3) by group 0's first thread once all of group 0 is done with chunk c -- group 1 then is, too.
  constexpr bool VST = PL::VST;
  auto vfetch = [&](int c) {                                   // G == 0: aux / addv rows completed by chunk c -> Vs[c & 1]
    if (c < k.nchunks) {
      const int jc0 = k.jlo + c * JC;
      cplx* vb = k.Vs + (size_t)(c & 1) * 2 * JC * AP_NC + k.tid;
#pragma unroll
      for (int r = 0; r < JC; ++r) {
        const int i = jc0 + r - W;
        if (i >= k.i0 && i < k.i1 && k.lane_ok) {
          if (p.aux) cp_async16(vb + r * AP_NC, p.aux + (size_t)i * ld + k.a);
          cp_async16(vb + (JC + r) * AP_NC, p.addv + (size_t)i * ld + k.a);
        }
      }
    }
    cp_async_commit();
  };
  if (G == 0 && VST) vfetch(0);
  for (int c = 0; c < k.nchunks; ++c) {
    const cplx* st = k.stage_base + (size_t)(c % PL::NSTAGE) * PL::STAGE;
    cplx* ps = k.Ps + (size_t)(c & 1) * JC * AP_NC;
    const cplx* vs = k.Vs + (size_t)(c & 1) * 2 * JC * AP_NC + k.tid;
    const int jc0 = k.jlo + c * JC;
    const int nr_real = min(JC, k.jhi - jc0);               // rows with data; later rows of the chunk are virtual
    const int nr_all = min(JC, k.jend - jc0);
    if (G == 0 && VST) { vfetch(c + 1); cp_async_wait<1>(); }
    if (nr_real > 0) mbar_wait(&k.full[c % PL::NSTAGE], (c / PL::NSTAGE) & 1);
    if (SPLIT && G == 1 && c >= 2) mbar_wait(&k.pempty[c & 1], ((c >> 1) - 1) & 1);
    if (SPLIT && G == 0) mbar_wait(&k.pfull[c & 1], (c >> 1) & 1);
#pragma unroll RU
    for (int r = 0; r < nr_all; ++r) {
      const int i = jc0 + r - W;                            // the output row completed by input row jc0 + r
      const bool emit = (G == 0) && (i >= k.i0) && k.lane_ok;
      cplx ax = make_double2(0, 0), pg = make_double2(0, 0);
      if (G == 0) {
        if (VST) {
          if (emit && p.aux) ax = vs[r * AP_NC];
        } else {
          if (emit && p.aux) ax = p.aux[(size_t)i * ld + k.a];
        }
        if (SPLIT) pg = ps[r * AP_NC + k.tid];
        if (VST && emit) pg = cadd(pg, vs[(JC + r) * AP_NC]);   // block part replaced by a known vector
      }
      if (r < nr_real) {
        const cplx* xs = st + PL::RS + PL::BS + (size_t)r * XW + k.tid + MAXM;
        if (G == 0 && BLK) {
          const cplx x0 = xs[0];
          if (k.slot >= 0) {
            const cplx* bc = st + PL::RS + ((size_t)k.slot * JC + r) * ND;
#pragma unroll
            for (int e = 0; e < ND; ++e) cfma(yw[e], bc[e], x0);
          } else {
            const cplx* bc = k.blk_g + (size_t)(jc0 + r) * ND;
#pragma unroll
            for (int e = 0; e < ND; ++e) cfma(yw[e], __ldg(bc + e), x0);
          }
        }
        if (T > 0 && GM > 0) {
          cplx z[T > 0 ? T : 1];
#pragma unroll
          for (int L = 0; L < T; ++L) z[L] = make_double2(0, 0);
#pragma unroll
          for (int o = -GM; o <= GM; ++o) {
            if (o == 0) continue;
            const cplx xo = xs[o];
#pragma unroll
            for (int L = 0; L < T; ++L) {
              if (PL::mine(G, L) && SH::m(L) >= (o < 0 ? -o : o)) {
                // slot order within a term: o = -m..-1 -> q = o + m ; o = 1..m -> q = m + o - 1
                const int q = o < 0 ? o + SH::m(L) : SH::m(L) + o - 1;
                if (L == LW) cfma(z[L], As[q * AP_NC], xo);
                else cfma(z[L], Areg[SH::slot0(L) + q], xo);
              }
            }
          }
#pragma unroll
          for (int L = 0; L < T; ++L) {
            if (!PL::mine(G, L)) continue;
            const cplx* rc = st + ((size_t)r * T + L) * ND;  // warp-uniform: broadcast LDS.128
#pragma unroll
            for (int e = 0; e < ND; ++e) cfma(yw[e], rc[e], z[L]);
          }
        }
      }
      if (G == 1) {
        if (SPLIT) ps[r * AP_NC + k.tid] = yw[0];
      } else if (emit) {
        cplx yv = cadd(yw[0], pg);
        if (p.emode == 2) {                                 // ||b||^2 = ||S c + r0 / 2||^2, nothing stored
          yv.x = fma(0.5, ax.x, yv.x); yv.y = fma(0.5, ax.y, yv.y);
        } else {
          if (p.emode == 1) { yv = cmul(p.oscale, yv); p.y2[(size_t)i * ld + k.a] = yv; }
          p.y[(size_t)i * ld + k.a] = yv;
          cfma_conj(d0, ax, yv);
        }
        d1 = fma(yv.x, yv.x, d1); d1 = fma(yv.y, yv.y, d1);
      }
#pragma unroll
      for (int e = 0; e < ND - 1; ++e) yw[e] = yw[e + 1];
      yw[ND - 1] = make_double2(0, 0);
    }
    if (G == 1) {
      if (SPLIT) mbar_arrive(&k.pfull[c & 1]);
    } else {
      if (SPLIT) mbar_arrive(&k.pempty[c & 1]);
      asm volatile("bar.sync 1, %0;" ::"n"(AP_NC) : "memory");   // group 0 only: everybody is done with stage c % NSTAGE
      if (k.tid == 0 && c + PL::NSTAGE < k.nchunks) issue(c + PL::NSTAGE);
    }
  }
  if (G == 0 && VST) cp_async_wait<0>();
}

template <int T, int M0, int MS, int W, int NG, bool BLK>
__global__ void __launch_bounds__(NG * AP_NC, (NG == 2 ? TDDE_AP_MINB2 : AP_MINB)) k_apply_banded(const __grid_constant__ ApplyArgs p) {
  using PL = ApplyPlan<T, M0, MS, W, NG, BLK>;
  constexpr int AP_BT = NG * AP_NC;
  constexpr int ND = PL::ND, MAXM = PL::MAXM, XW = PL::XW, JC = PL::JC;
  if (p.guard == 1 && solver_idle(p.red.st)) return;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  ApplyCommon k;
  k.stage_base = reinterpret_cast<cplx*>(smem_raw);
  k.Ps = k.stage_base + (size_t)PL::NSTAGE * PL::STAGE;
  k.Vs = k.Ps + PL::PS;
  k.As = k.Vs + PL::VS;
  k.full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)(PL::NSTAGE * PL::STAGE + PL::PS + PL::VS + PL::AS) * sizeof(cplx));
  k.pfull = k.full + PL::NSTAGE;
  k.pempty = k.pfull + 2;

  const int grp = threadIdx.x / AP_NC;                       // warp-uniform
  k.tid = threadIdx.x % AP_NC;
  const int a0 = blockIdx.x * AP_NC;
  k.a = a0 + k.tid;                                          // channel; lanes with a >= ld idle along
  k.ld = p.ld; k.n_rad = p.n_rad;
  k.lane_ok = k.a >= p.own_lo && k.a < p.own_hi;              // own_hi <= ld
  k.ac = k.a < k.ld ? k.a : k.ld - 1;
  k.i0 = blockIdx.y * p.seg_len;
  k.i1 = min(k.n_rad, k.i0 + p.seg_len);
  k.jlo = max(0, k.i0 - W);
  k.jhi = min(k.n_rad, k.i1 + W);                            // input rows [jlo, jhi) carry data
  k.jend = k.i1 + W;                                         // rows [jhi, jend) only flush the output window
  k.nchunks = (k.jend - k.jlo + JC - 1) / JC;
  k.slot = p.slot[k.ac];                                     // index into this CTA's class list, or -1
  k.blk_g = p.blk + (size_t)p.cls[k.ac] * k.n_rad * ND;      // global fallback for slot < 0

  // channel range of the x tile, clipped to the vector; the clipped cells stay zero (matching A entries are 0)
  const int ld = k.ld, n_rad = k.n_rad, jlo = k.jlo, jhi = k.jhi;
  const int xa_lo = max(0, a0 - MAXM), xa_hi = min(ld, a0 + AP_NC + MAXM);
  const int x_dst_off = xa_lo - (a0 - MAXM);
  const uint32_t x_bytes = (uint32_t)(xa_hi - xa_lo) * sizeof(cplx);
  const int* cta_cls = p.cta_cls + blockIdx.x * AP_MAXC;
  cplx* stage_base = k.stage_base;
  uint64_t* full = k.full;

  if (x_bytes != XW * sizeof(cplx)) {
    for (int q = threadIdx.x; q < PL::NSTAGE * PL::STAGE; q += AP_BT) stage_base[q] = make_double2(0, 0);
  }
  if (threadIdx.x == 0) {
    for (int q = 0; q < PL::NSTAGE; ++q) mbar_init(&full[q], 1);
    for (int q = 0; q < 2; ++q) { mbar_init(&k.pfull[q], AP_NC); mbar_init(&k.pempty[q], AP_NC); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");

  auto issue = [&](int c) {                                  // one elected thread: all bulk copies of chunk c
    cplx* st = stage_base + (size_t)(c % PL::NSTAGE) * PL::STAGE;
    uint64_t* bar = &full[c % PL::NSTAGE];
    const int j = jlo + c * JC;
    const int nr = min(JC, jhi - j);
    if (nr <= 0) return;                                     // a chunk of virtual rows only
    const bool x2d = (T == 0) && p.use_xmap;                  // one tensor copy: full box, out-of-bounds zero-filled
    uint32_t bytes = x2d ? (uint32_t)(JC * AP_NC * sizeof(cplx)) : (uint32_t)nr * x_bytes;
    int ncls = 0;
    if (BLK) {
#pragma unroll
      for (int q = 0; q < AP_MAXC; ++q) ncls += (cta_cls[q] >= 0);
    }
    bytes += (uint32_t)ncls * nr * ND * sizeof(cplx);
    if (T > 0) bytes += (uint32_t)nr * T * ND * sizeof(cplx);
    mbar_expect_tx(bar, bytes);
    if (T > 0) bulk_g2s(st, p.Rall + (size_t)j * T * ND, (uint32_t)nr * T * ND * sizeof(cplx), bar);
#pragma unroll
    for (int q = 0; q < AP_MAXC; ++q) {
      const int kk = BLK ? cta_cls[q] : -1;
      if (kk >= 0)
        bulk_g2s(st + PL::RS + (size_t)q * JC * ND, p.blk + ((size_t)kk * n_rad + j) * ND, (uint32_t)nr * ND * sizeof(cplx), bar);
    }
    if (x2d) {
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                       smem_u32(st + PL::RS + PL::BS)),
                   "l"(reinterpret_cast<uint64_t>(&p.xmap)), "r"(2 * a0), "r"(j), "r"(smem_u32(bar))
                   : "memory");
    } else {
      for (int r = 0; r < nr; ++r)
        bulk_g2s(st + PL::RS + PL::BS + (size_t)r * XW + x_dst_off, p.x + (size_t)(j + r) * ld + xa_lo, x_bytes, bar);
    }
  };
  if (threadIdx.x == 0) {
    for (int c = 0; c < PL::NSTAGE && c < k.nchunks; ++c) issue(c);
  }

  cplx d0 = make_double2(0, 0);
  double d1 = 0;
  if (NG == 1 || grp == 0) apply_group<T, M0, MS, W, NG, BLK, 0>(p, k, issue, d0, d1);
  else apply_group<T, M0, MS, W, NG, BLK, 1>(p, k, issue, d0, d1);
  if (p.red.fin != FIN_NONE) grid_reduce_finalize<AP_BT>(d0.x, d0.y, d1, p.red);
}

// ---- generic path: arbitrary CSR A_L, arbitrary per-term bandwidths; one thread per output element, no staging. ----
// Correct for any input the ABI accepts; the fall-back when neither structured kernel applies.  The grid is bounded
// (blocks stride over (row, channel-block) pairs), so the per-block reduction scratch can never overflow.
__global__ void __launch_bounds__(AP_NT) k_apply_generic(const ApplyArgs p) {
  if (p.guard == 1 && solver_idle(p.red.st)) return;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;
  const int ld = p.ld, n_rad = p.n_rad;
  const int cb = (ld + AP_NT - 1) / AP_NT;
  const long long nwork = (long long)cb * n_rad;
  cplx d0 = make_double2(0, 0);
  double d1 = 0;
  for (long long wk = blockIdx.x; wk < nwork; wk += gridDim.x) {
    const int a = (int)(wk % cb) * AP_NT + threadIdx.x;
    const int i = (int)(wk / cb);
    if (a >= p.own_hi || a < p.own_lo) continue;
    cplx acc = make_double2(0, 0);
    if (a < p.n_ang) {
      const int w0 = p.w0, nd0 = 2 * w0 + 1;
      const cplx* br = p.blk_row + ((size_t)p.cls[a] * n_rad + i) * nd0;
      for (int d = -w0; d <= w0; ++d) {
        const int j = i + d;
        if (j >= 0 && j < n_rad) cfma(acc, br[d + w0], p.x[(size_t)j * ld + a]);
      }
      const double* g = p.g + (p.step_ptr ? (size_t)(*p.step_ptr) * p.n_terms : 0);
      for (int L = 0; L < p.n_terms; ++L) {
        const double gl = g[L];
        if (gl == 0.0) continue;
        const int w = p.w[L], nd = 2 * w + 1;
        const cplx* rr = p.Rrow[L] + (size_t)i * nd;
        cplx tsum = make_double2(0, 0);
        for (int q = p.A_rowptr[L][a]; q < p.A_rowptr[L][a + 1]; ++q) {
          const int ca = p.A_col[L][q];
          cplx rs = make_double2(0, 0);
          for (int d = -w; d <= w; ++d) {
            const int j = i + d;
            if (j >= 0 && j < n_rad) cfma(rs, rr[d + w], p.x[(size_t)j * ld + ca]);
          }
          cfma(tsum, p.A_val[L][q], rs);
        }
        cfma(acc, make_double2(p.beta.x * gl, p.beta.y * gl), tsum);
      }
    }
    if (p.emode == 2) {
      const cplx ax = p.aux[(size_t)i * ld + a];
      acc.x = fma(0.5, ax.x, acc.x); acc.y = fma(0.5, ax.y, acc.y);
    } else {
      if (p.emode == 1) { acc = cmul(p.oscale, acc); p.y2[(size_t)i * ld + a] = acc; }
      p.y[(size_t)i * ld + a] = acc;
      if (p.aux) cfma_conj(d0, p.aux[(size_t)i * ld + a], acc);
    }
    d1 = fma(acc.x, acc.x, d1); d1 = fma(acc.y, acc.y, d1);
  }
  if (p.red.fin != FIN_NONE) grid_reduce_finalize<AP_NT>(d0.x, d0.y, d1, p.red);
}

// ---- instantiation registry ----
#define TDDE_BANDED_SHAPES(X) \
  X(0, 0, 0, 3) X(0, 0, 0, 6) X(0, 0, 0, 9) \
  X(1, 1, 1, 3) X(2, 1, 1, 3) X(3, 2, 0, 3) \
  X(5, 1, 1, 6) \
  X(7, 1, 1, 3) X(7, 1, 1, 6) X(7, 1, 1, 9)

// the instantiated shapes (T, M0, MS, W), for the structure fit at create
int apply_banded_shapes(int (*out)[4], int cap) {
  int n = 0;
#define X(t, a, b, w) if (n < cap) { out[n][0] = t; out[n][1] = a; out[n][2] = b; out[n][3] = w; ++n; }
  TDDE_BANDED_SHAPES(X)
#undef X
  return n;
}

bool apply_banded_available(int T, int m0, int mstep, int W) {
#define X(t, a, b, w) if (T == t && (t == 0 || (m0 == a && mstep == b)) && W == w) return true;
  TDDE_BANDED_SHAPES(X)
#undef X
  return false;
}

template <int T, int M0, int MS, int W, int NG, bool BLK>
static int launch_banded_one(const ApplyArgs& a, dim3 grid, cudaStream_t s) {
  static bool attr_set[64] = {};                            // per device: the attribute belongs to the function on one device
  const size_t smem = ApplyPlan<T, M0, MS, W, NG, BLK>::SMEM;
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || !attr_set[dev]) {
    if (cudaFuncSetAttribute(k_apply_banded<T, M0, MS, W, NG, BLK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
        cudaSuccess)
      return -2;
    if (dev >= 0 && dev < 64) attr_set[dev] = true;
  }
  k_apply_banded<T, M0, MS, W, NG, BLK><<<grid, NG * AP_NC, smem, s>>>(a);
  return 1;
}

// ng = number of warp groups the terms of a channel are split over (1 or 2); T == 0 always runs with one group.
int launch_apply_banded(const ApplyArgs& a, int T, int m0, int mstep, int W, int ng, cudaStream_t s) {
  dim3 grid((a.ld + AP_NC - 1) / AP_NC, (a.n_rad + a.seg_len - 1) / a.seg_len);
#define X(t, aa, b, w)                                                          \
  if (T == t && (t == 0 || (m0 == aa && mstep == b)) && W == w) {               \
    if (t == 0) return launch_banded_one<t, aa, b, w, 1, true>(a, grid, s);                                      \
    if (a.addv) return ng == 1 ? launch_banded_one<t, aa, b, w, 1, (t == 0)>(a, grid, s)                         \
                               : launch_banded_one<t, aa, b, w, (t == 0 ? 1 : 2), (t == 0)>(a, grid, s);         \
    return ng == 1 ? launch_banded_one<t, aa, b, w, 1, true>(a, grid, s)                                         \
                   : launch_banded_one<t, aa, b, w, (t == 0 ? 1 : 2), true>(a, grid, s);                         \
  }
  TDDE_BANDED_SHAPES(X)
#undef X
  return -1;
}

int launch_apply_generic(const ApplyArgs& a, int num_sms, cudaStream_t s) {
  const long long nwork = (long long)((a.ld + AP_NT - 1) / AP_NT) * a.n_rad;
  const long long cap = std::min<long long>((long long)num_sms * 16, TDDE_MAX_PARTIAL_BLOCKS);
  const int grid = (int)std::max<long long>(1, std::min(nwork, cap));
  k_apply_generic<<<grid, AP_NT, 0, s>>>(a);
  return 1;
}
