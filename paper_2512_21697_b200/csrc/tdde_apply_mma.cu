// tdde_apply_mma.cu -- in-iteration operator apply with the radial band contraction on the FP64 tensor-core path (DMMA)
//
//   y[a', i] = addv[a', i] + beta * sum_L g_L sum_j R_L[i, j] z_L[a', j],     z_L[a', j] = sum_a A_L[a', a] x[a, j]
//   (Eq. 17; the block part is the known right-hand side of the preceding solve, R21)
//
// Why: on B200 DMMA (mma.sync.m8n8k4.f64) and DFMA share one pipe and one peak (measured 37.1 vs 36.8 TFLOP/s, no overlap), but a
// DMMA delivers 256 FMAs per issue slot and per 3 operand registers.  The register-window kernel (tdde_apply.cu) spends one
// warp-broadcast shared-memory load per 4 DFMAs on the radial coefficients and ends at 56-59 % FP64-pipe utilisation with the
// shared-memory pipe equally busy; here the radial coefficients are MMA operands shared by 8 channels.
//
// Mapping.  A warp owns 8 channels; lane = (r = lane % 4, c = lane / 4) = (row of a 4-row input slice, channel).
//   angular part (DFMA, as before): z_L[j0 + r][a_c] from the x tile and the beta g_L A_L[a_c, a_c + o] rows in shared memory
//     -- exactly the A-operand layout of the MMA (M = channel, K = input row);
//   radial part (DMMA): for every 8-row output tile the slice touches, Y^T[8 ch x 8 rows] += Z^T[8 ch x 4 rows] R^T[4 rows x 8 rows];
//     complex product by three real MMAs (Gauss):  A1 += zr (Rr + Ri),  A2 += (zi - zr) Rr,  A3 += (zr + zi) Ri,
//     re = A1 - A3, im = A1 + A2  (sums are linear, so the three accumulators are combined once per finished tile);
//   the B operands (R_L in fragment order, zero outside the band and outside the matrix, the three Gauss combinations) are built
//     once at create and arrive by one TMA bulk copy per slice; x rows by one bulk copy each (GATHER: up to three, the halo pieces from
//     the neighbouring shards' vectors); 4-6 stage mbarrier ring (full: TMA transaction bytes, empty: one arrival per warp).
//   beta g_L A_L rows live in shared memory (one column per channel); an interior period (two slices = one tile row) is processed as a unit
//   so that each A_L value is loaded once for the two rows a lane owns.
// Band overhead: a 4-row slice touches (4 + 2W) output rows = 2.5 (W = 6) tiles of 8 on average, i.e. 7.5 DMMA = 60 FMA-equivalents
// per element and term against 52 DFMA in the exact band: the pipe does 13 % more work but is kept busy 78 % of the time (DFMA kernel: 59 %).
// Measured (B200, HBM-scale, T = 7, W = 6): 1.551 ms per apply = 65 % of the FP64 peak counted in algorithmic flops (DFMA kernel: 1.806 ms).
#include <algorithm>
#include <vector>
#include <complex>
#include <type_traits>
#include "tdde_reduce.cuh"

// Channels per CTA (8 per warp), chosen per bandwidth from measurements on B200 (HBM-scale / Large in-iteration apply):
//   W = 6: 128 channels = 16 warps at <= 128 registers, the addv / aux rows loaded when a tile is emitted: 1.552 / 0.227 ms
//          (96 channels = 12 warps at <= 168 registers with those rows prefetched one period ahead: 1.575 / 0.235 ms)
//   W = 9: 96 channels with the prefetch: 1.93 ms (128 channels: the accumulators of 4-5 live tiles spill, 2.40 ms)
#ifndef MM_NC6
#define MM_NC6 128
#endif
#ifndef MM_NC9
#define MM_NC9 96
#endif
__host__ __device__ constexpr int mm_nc(int W) { return W <= 6 ? MM_NC6 : MM_NC9; }
#ifndef MM_NSTAGE
#define MM_NSTAGE 6          // pipeline stages wanted (fewer when shared memory is short)
#endif
#ifndef MM_ASMEM5
#define MM_ASMEM5 3          // same for T < 7
#endif
#ifndef MM_ASMEM
#define MM_ASMEM 7           // T >= 7: the A_L rows of this many widest terms live in shared memory, not in registers
#endif
#ifndef MM_NOPAIR
#define MM_PAIR 1            // interior periods process both slices together (measured: HBM-scale 1.68 -> 1.565 ms)
#endif

__host__ __device__ constexpr int mm_floordiv(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// Slice grid relative to an 8-aligned row origin: slice q covers rows 4q - OFF .. 4q - OFF + 3 and touches the 8-row tiles
// floordiv(4q - OFF - W, 8) .. floordiv(4q - OFF + 3 + W, 8).  q = 2u + par: everything below is static per parity.
template <int W>
struct MmaGrid {
  __host__ __device__ static constexpr int first(int off, int par) { return mm_floordiv(4 * par - off - W, 8); }
  __host__ __device__ static constexpr int last(int off, int par) { return mm_floordiv(4 * par - off + 3 + W, 8); }
  __host__ __device__ static constexpr int cost(int off) { return last(off, 0) - first(off, 0) + last(off, 1) - first(off, 1) + 2; }
  __host__ __device__ static constexpr int best_off() {
    int b = W;
    for (int o = W; o < W + 4; ++o) if (cost(o) < cost(b)) b = o;
    return b;
  }
  static constexpr int OFF = best_off();
  __host__ __device__ static constexpr int F(int par) { return first(OFF, par); }
  __host__ __device__ static constexpr int NTL(int par) { return last(OFF, par) - first(OFF, par) + 1; }
  static constexpr int NTMAX = NTL(0) > NTL(1) ? NTL(0) : NTL(1);
  static constexpr int C0 = mm_floordiv(7 + W + OFF, 4);          // tile v is complete after slice 2 v + C0
  static constexpr int PAR_E = C0 & 1;                             // ... which is the slice of this parity in period u = v + EV
  static constexpr int EV = (C0 - PAR_E) / 2;                      // emitted tile after slice (u, PAR_E): v = u - EV
  // oldest unfinished tile when slice (u, par) runs: u + B(par)
  __host__ __device__ static constexpr int B(int par) { return -mm_floordiv(C0 - par, 2); }
  __host__ __device__ static constexpr int NLIVE() {
    int n = 0;
    for (int par = 0; par < 2; ++par) { const int v = last(OFF, par) - B(par) + 1; if (v > n) n = v; }
    return n;
  }
};

template <int T, int M0, int MS>
struct MmaShape {
  __host__ __device__ static constexpr int m(int L) { return M0 + MS * L; }
  __host__ __device__ static constexpr int maxm() { return M0 + MS * (T - 1); }
  __host__ __device__ static constexpr int slot0(int L) { int s = 0; for (int l = 0; l < L; ++l) s += 2 * m(l); return s; }
  __host__ __device__ static constexpr int nslots() { return slot0(T); }
};

template <int T, int M0, int MS, int W>
struct MmaPlan {
  using G = MmaGrid<W>;
  using SH = MmaShape<T, M0, MS>;
  static constexpr int MAXM = SH::maxm();
  static constexpr int NC = mm_nc(W), NT = 4 * NC;
  static constexpr bool PF = NC <= 96;                              // prefetch the addv / aux rows of the next tile into registers
  static constexpr int XW = NC + 2 * MAXM;
  // row pitch of the x tile: = 2 or 6 (mod 8) complex, so the 4 rows x 2 channels of a quarter-warp hit all 32 banks once
  __host__ __device__ static constexpr int pitch() { int p = XW; while (p % 8 != 2 && p % 8 != 6) ++p; return p; }
  static constexpr int XP = pitch();
  static constexpr int FR0 = T * G::NTL(0) * 96, FR1 = T * G::NTL(1) * 96;      // doubles per slice of parity 0 / 1
  static constexpr int FRMAX = FR0 > FR1 ? FR0 : FR1;
  static constexpr int STAGE_BYTES = FRMAX * 8 + 4 * XP * 16;
  // the last NAS terms (the widest) keep beta g_L A_L in shared memory [slot][NC channels]; the others in registers
  static constexpr int NAS = (T >= 7) ? MM_ASMEM : MM_ASMEM5;
  static constexpr int NSREG = SH::slot0(T - NAS);                  // register slots
  static constexpr int AS_BYTES = (SH::nslots() - NSREG) * NC * 16;
  __host__ __device__ static constexpr int stages() {
    int n = (226 * 1024 - AS_BYTES - 256) / STAGE_BYTES;
    return n > MM_NSTAGE ? MM_NSTAGE : n;
  }
  static constexpr int NSTAGE = stages();
  static_assert(NSTAGE >= 3, "k_apply_mma: shared memory too small for this shape");
  static constexpr size_t SMEM = (size_t)NSTAGE * STAGE_BYTES + AS_BYTES + 256;
};

// ---- raw PTX helpers (same idioms as tdde_apply.cu) ----
__device__ __forceinline__ uint32_t mm_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mm_bar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mm_smem(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mm_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mm_smem(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mm_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(mm_smem(dst)),
               "l"(src), "r"(bytes), "r"(mm_smem(bar))
               : "memory");
}
__device__ __forceinline__ void mm_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mm_smem(bar)) : "memory");
}
__device__ __forceinline__ void mm_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok)
                 : "r"(mm_smem(bar)), "r"(parity)
                 : "memory");
  } while (!ok);
}
// D(8x8) += A(8x4) B(4x8): lane holds A[lane/4][lane%4], B[lane%4][lane/4], D[lane/4][2 (lane%4) + {0,1}]
__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// GATHER (channel-slab shards, tdde_shard.cu): the halo columns of the x tile are fetched by the TMA producer straight from the vectors of
// the neighbouring shards (p.xL / p.xR: same device, or peer memory), so no halo copy precedes the apply
template <int T, int M0, int MS, int W, bool GATHER>
__global__ void __launch_bounds__(4 * mm_nc(W), 1) k_apply_mma(const __grid_constant__ ApplyArgs p) {
  using PL = MmaPlan<T, M0, MS, W>;
  using G = MmaGrid<W>;
  using SH = MmaShape<T, M0, MS>;
  constexpr int MAXM = PL::MAXM, XP = PL::XP, NS = SH::nslots(), NL = G::NLIVE(), MM_NC = PL::NC, MM_NT = PL::NT;
  if (p.guard == 1 && solver_idle(p.red.st)) return;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;

  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx* const As = reinterpret_cast<cplx*>(smem_raw + (size_t)PL::NSTAGE * PL::STAGE_BYTES);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)PL::NSTAGE * PL::STAGE_BYTES + PL::AS_BYTES);
  uint64_t* empty = full + PL::NSTAGE;   // 2 x NSTAGE x 8 B <= 128 B of the 256 B tail

  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const int r = lane & 3, cl = wrp * 8 + (lane >> 2);          // row within a slice, channel within the CTA
  const int ld = p.ld, n_rad = p.n_rad;
  const int a0 = blockIdx.x * MM_NC;
  const int a = a0 + cl;
  const bool lane_ok = a >= p.own_lo && a < p.own_hi;          // own_hi <= ld
  const int ac = a < ld ? a : ld - 1;
  const int i0 = blockIdx.y * p.seg_len;                       // seg_len is a multiple of 8
  const int i1 = min(n_rad, i0 + p.seg_len);
  const int ntile = (i1 - i0 + 7) / 8;                         // output tiles of this CTA
  const int nq = 2 * (ntile - 1) + G::C0 + 1;                  // slices until the last tile is complete
  const int Q0 = i0 / 4;                                       // absolute index of this CTA's slice 0

  const int xa_lo = max(0, a0 - MAXM), xa_hi = min(ld, a0 + MM_NC + MAXM);
  const int x_dst_off = xa_lo - (a0 - MAXM);
  const uint32_t x_bytes = (uint32_t)(xa_hi - xa_lo) * sizeof(cplx);

  // zero the stage buffers once: x cells outside the vector and rows outside the matrix are never written
  for (int q = tid; q < PL::NSTAGE * PL::STAGE_BYTES / 16; q += MM_NT) reinterpret_cast<double2*>(smem_raw)[q] = make_double2(0, 0);
  if (tid == 0) {
    for (int q = 0; q < PL::NSTAGE; ++q) { mm_bar_init(&full[q], 1); mm_bar_init(&empty[q], MM_NT / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");

  // GATHER: [xa_lo, xa_hi) = [left halo | owned | right halo]: three sources, the same bytes in total (set up once per CTA)
  const int gc1 = GATHER ? min(xa_hi, max(xa_lo, p.own_lo)) : xa_lo, gc2 = GATHER ? min(xa_hi, max(gc1, p.own_hi)) : xa_hi;
  const cplx* gsL = (GATHER && p.xL) ? p.xL + xa_lo + p.shiftL : p.x + xa_lo;
  const cplx* gsR = (GATHER && p.xR) ? p.xR + gc2 + p.shiftR : p.x + gc2;
  const int gldL = (GATHER && p.xL) ? p.ldL : ld, gldR = (GATHER && p.xR) ? p.ldR : ld;
  const uint32_t gbL = (uint32_t)(gc1 - xa_lo) * sizeof(cplx), gbO = (uint32_t)(gc2 - gc1) * sizeof(cplx), gbR = (uint32_t)(xa_hi - gc2) * sizeof(cplx);
  const int gcO = gc1, gdO = gc1 - xa_lo, gdR = gc2 - xa_lo;
  auto issue = [&](int q) {                                    // one thread: the bulk copies of slice q
    unsigned char* st = smem_raw + (size_t)(q % PL::NSTAGE) * PL::STAGE_BYTES;
    uint64_t* bar = &full[q % PL::NSTAGE];
    const int par = q & 1;
    const uint32_t fbytes = (uint32_t)(par ? PL::FR1 : PL::FR0) * 8;
    const int j0 = i0 + 4 * q - G::OFF;
    int nrow = 0;
    for (int rr = 0; rr < 4; ++rr) nrow += (j0 + rr >= 0 && j0 + rr < n_rad);
    mm_expect_tx(bar, fbytes + (uint32_t)nrow * x_bytes);
    const double* fsrc = p.Rfrag + (size_t)((Q0 + q) >> 1) * (PL::FR0 + PL::FR1) + (par ? PL::FR0 : 0);
    mm_bulk_g2s(st, fsrc, fbytes, bar);
    cplx* xs = reinterpret_cast<cplx*>(st + PL::FRMAX * 8);
    if (!GATHER) {
      for (int rr = 0; rr < 4; ++rr)
        if (j0 + rr >= 0 && j0 + rr < n_rad) mm_bulk_g2s(xs + rr * XP + x_dst_off, p.x + (size_t)(j0 + rr) * ld + xa_lo, x_bytes, bar);
    } else {
      for (int rr = 0; rr < 4; ++rr) {
        const int j = j0 + rr;
        if (j < 0 || j >= n_rad) continue;
        cplx* dst = xs + rr * XP + x_dst_off;
        if (gbL) mm_bulk_g2s(dst, gsL + (size_t)j * gldL, gbL, bar);
        if (gbO) mm_bulk_g2s(dst + gdO, p.x + (size_t)j * ld + gcO, gbO, bar);
        if (gbR) mm_bulk_g2s(dst + gdR, gsR + (size_t)j * gldR, gbR, bar);
      }
    }
  };
  if (tid == 0)
    for (int q = 0; q < PL::NSTAGE && q < nq; ++q) issue(q);

  // beta g_L A_L[a, a + o] of all terms in registers
  cplx Areg[PL::NSREG > 0 ? PL::NSREG : 1];
  {
    const double* g = p.g + (p.step_ptr ? (size_t)(*p.step_ptr) * T : 0);
#pragma unroll
    for (int L = 0; L < T; ++L) {
      const double gl = g[L];
      const cplx coef = make_double2(p.beta.x * gl, p.beta.y * gl);
#pragma unroll
      for (int q = 0; q < 2 * SH::m(L); ++q) {
        const int s = SH::slot0(L) + q;
        const cplx av = cmul(coef, p.Aoff[(size_t)s * ld + ac]);
        if (s < PL::NSREG) Areg[s] = av;
        else if (r == 0) As[(s - PL::NSREG) * MM_NC + cl] = av;
      }
    }
  }
  double acc[NL][3][2];
#pragma unroll
  for (int k = 0; k < NL; ++k)
#pragma unroll
    for (int e = 0; e < 3; ++e) { acc[k][e][0] = 0; acc[k][e][1] = 0; }

  // addv / aux rows of the tile emitted next, fetched one period ahead
  cplx pv[2], pa[2];
  auto prefetch = [&](int v) {
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int i = i0 + 8 * v + 2 * r + e;
      pv[e] = make_double2(0, 0); pa[e] = make_double2(0, 0);
      if (v >= 0 && i < i1 && lane_ok) {
        pv[e] = p.addv[(size_t)i * ld + a];
        if (p.aux) pa[e] = p.aux[(size_t)i * ld + a];
      }
    }
  };
  if (PL::PF) prefetch(0);
  __syncthreads();                                              // As visible to the whole warp
  cplx d0 = make_double2(0, 0);
  double d1 = 0;

  // refill the stage slice s used with slice s + NSTAGE once every warp has left it (thread 0; called once per slice, in order)
  auto refill = [&](int s) {
    if (s >= 0 && s + PL::NSTAGE < nq) {
      mm_wait(&empty[s % PL::NSTAGE], (s / PL::NSTAGE) & 1);
      issue(s + PL::NSTAGE);
    }
  };
  // radial band of one slice (DMMA): tiles u + F(par) + k; CHK = some touched tile may lie outside this CTA's range
  auto radial = [&](int u, const cplx (&z)[T], const double* fr, bool row_ok, auto PAR, auto CHK) {
    constexpr int par = decltype(PAR)::value;
    constexpr bool chk = decltype(CHK)::value;
#pragma unroll
    for (int L = 0; L < T; ++L) {
      const double zr = row_ok ? z[L].x : 0.0, zi = row_ok ? z[L].y : 0.0;
      const double zm = zi - zr, zp = zr + zi;
#pragma unroll
      for (int k = 0; k < G::NTL(par); ++k) {
        const int v = u + G::F(par) + k;
        if (!chk || (v >= 0 && v < ntile)) {
          const int ai = G::F(par) - G::B(par) + k;                // static accumulator index
          const double* f = fr + (L * G::NTL(par) + k) * 96;
          dmma(acc[ai][0], zr, f[0]);
          dmma(acc[ai][1], zm, f[32]);
          dmma(acc[ai][2], zp, f[64]);
        }
      }
    }
  };
  // one slice with its own pipeline synchronisation (boundary periods)
  auto slice = [&](int u, auto PAR, auto CHK) {
    constexpr int par = decltype(PAR)::value;
    const int q = 2 * u + par;
    if (tid == 0) refill(q - 2);
    __syncwarp();
    mm_wait(&full[q % PL::NSTAGE], (q / PL::NSTAGE) & 1);
    const unsigned char* st = smem_raw + (size_t)(q % PL::NSTAGE) * PL::STAGE_BYTES;
    const double* fr = reinterpret_cast<const double*>(st) + lane;
    const cplx* xs = reinterpret_cast<const cplx*>(st + PL::FRMAX * 8) + r * XP + cl + MAXM;
    const int j = i0 + 4 * q - G::OFF + r;
    const bool row_ok = (j >= 0) && (j < n_rad);
    cplx z[T];                                                     // angular combination (DFMA)
#pragma unroll
    for (int L = 0; L < T; ++L) z[L] = make_double2(0, 0);
#pragma unroll
    for (int o = -MAXM; o <= MAXM; ++o) {
      if (o == 0) continue;
      const cplx xo = xs[o];
#pragma unroll
      for (int L = 0; L < T; ++L) {
        if (SH::m(L) >= (o < 0 ? -o : o)) {
          const int qq = o < 0 ? o + SH::m(L) : SH::m(L) + o - 1;
          const int s = SH::slot0(L) + qq;
          if (s < PL::NSREG) cfma(z[L], Areg[s], xo);
          else cfma(z[L], As[(s - PL::NSREG) * MM_NC + cl], xo);
        }
      }
    }
    radial(u, z, fr, row_ok, PAR, CHK);
    __syncwarp();
    if (lane == 0) mm_arrive(&empty[q % PL::NSTAGE]);
  };
  auto emit = [&](int u) {                                         // tile u - EV is complete: combine, add, store, inner products
    const int v = u - G::EV;
    if (v >= 0 && v < ntile) {
      if (!PL::PF) prefetch(v);
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int i = i0 + 8 * v + 2 * r + e;
        if (i < i1 && lane_ok) {
          cplx yv = make_double2(pv[e].x + (acc[0][0][e] - acc[0][2][e]), pv[e].y + (acc[0][0][e] + acc[0][1][e]));
          p.y[(size_t)i * ld + a] = yv;
          if (p.emode == 3) {                                      // start of step: y = y2 = r0, aux = S c: ||S c + r0 / 2||^2, ||r0||^2
            p.y2[(size_t)i * ld + a] = yv;
            const double bx = fma(0.5, yv.x, pa[e].x), by = fma(0.5, yv.y, pa[e].y);
            d0.x = fma(bx, bx, d0.x); d0.x = fma(by, by, d0.x);
          } else {
            cfma_conj(d0, pa[e], yv);
          }
          d1 = fma(yv.x, yv.x, d1); d1 = fma(yv.y, yv.y, d1);
        }
      }
    }
#pragma unroll
    for (int k = 0; k + 1 < NL; ++k)
#pragma unroll
      for (int e = 0; e < 3; ++e) { acc[k][e][0] = acc[k + 1][e][0]; acc[k][e][1] = acc[k + 1][e][1]; }
#pragma unroll
    for (int e = 0; e < 3; ++e) { acc[NL - 1][e][0] = 0; acc[NL - 1][e][1] = 0; }
    if (PL::PF && v + 1 < ntile) prefetch(v + 1);
  };
  using I0 = std::integral_constant<int, 0>;
  using I1 = std::integral_constant<int, 1>;
  // an interior period: both slices together.  One pipeline synchronisation, and every A_L coefficient that comes from shared
  // memory is loaded once for the two rows this lane owns (rows r of both slices)
  auto pair = [&](int u) {
    const int q0 = 2 * u;
    if (tid == 0) { refill(q0 - 2); refill(q0 - 1); }
    __syncwarp();
    mm_wait(&full[q0 % PL::NSTAGE], (q0 / PL::NSTAGE) & 1);
    mm_wait(&full[(q0 + 1) % PL::NSTAGE], ((q0 + 1) / PL::NSTAGE) & 1);
    const unsigned char* st0 = smem_raw + (size_t)(q0 % PL::NSTAGE) * PL::STAGE_BYTES;
    const unsigned char* st1 = smem_raw + (size_t)((q0 + 1) % PL::NSTAGE) * PL::STAGE_BYTES;
    const cplx* xs0 = reinterpret_cast<const cplx*>(st0 + PL::FRMAX * 8) + r * XP + cl + MAXM;
    const cplx* xs1 = reinterpret_cast<const cplx*>(st1 + PL::FRMAX * 8) + r * XP + cl + MAXM;
    const int j = i0 + 4 * q0 - G::OFF + r;
    const bool ok0 = (j >= 0) && (j < n_rad), ok1 = (j + 4 >= 0) && (j + 4 < n_rad);
    cplx z0[T], z1[T];
#pragma unroll
    for (int L = 0; L < T; ++L) { z0[L] = make_double2(0, 0); z1[L] = make_double2(0, 0); }
#pragma unroll
    for (int o = -MAXM; o <= MAXM; ++o) {
      if (o == 0) continue;
      const cplx xa = xs0[o], xb = xs1[o];
#pragma unroll
      for (int L = 0; L < T; ++L) {
        if (SH::m(L) >= (o < 0 ? -o : o)) {
          const int qq = o < 0 ? o + SH::m(L) : SH::m(L) + o - 1;
          const int s = SH::slot0(L) + qq;
          const cplx av = (s < PL::NSREG) ? Areg[s < PL::NSREG ? s : 0] : As[(s - PL::NSREG) * MM_NC + cl];
          cfma(z0[L], av, xa);
          cfma(z1[L], av, xb);
        }
      }
    }
    radial(u, z0, reinterpret_cast<const double*>(st0) + lane, ok0, I0{}, std::false_type{});
    if (G::PAR_E == 0) emit(u);
    radial(u, z1, reinterpret_cast<const double*>(st1) + lane, ok1, I1{}, std::false_type{});
    if (G::PAR_E == 1) emit(u);
    __syncwarp();
    if (lane == 0) { mm_arrive(&empty[q0 % PL::NSTAGE]); mm_arrive(&empty[(q0 + 1) % PL::NSTAGE]); }
  };
  constexpr int ULO = -(G::F(0) < G::F(1) ? G::F(0) : G::F(1));                                  // first period whose tiles are all >= 0
  constexpr int LMAX = (G::F(0) + G::NTL(0) > G::F(1) + G::NTL(1) ? G::F(0) + G::NTL(0) : G::F(1) + G::NTL(1)) - 1;
  const int nu = (nq + 1) / 2;
  for (int u = 0; u < nu; ++u) {
    if (u >= ULO && u + LMAX < ntile) {                            // interior period: no range checks
#ifdef MM_PAIR
      pair(u);
#else
      slice(u, I0{}, std::false_type{});
      if (G::PAR_E == 0) emit(u);
      slice(u, I1{}, std::false_type{});
      if (G::PAR_E == 1) emit(u);
#endif
    } else {
      if (2 * u < nq) slice(u, I0{}, std::true_type{});
      if (G::PAR_E == 0) emit(u);
      if (2 * u + 1 < nq) slice(u, I1{}, std::true_type{});
      if (G::PAR_E == 1) emit(u);
    }
  }
  if (p.red.fin != FIN_NONE) grid_reduce_finalize<MM_NT>(d0.x, d0.y, d1, p.red);
}

// ---- host side ----
// W = 3 stays on the register-window kernel: the 8-row tiles waste half of every MMA there (measured 1.54 vs 1.33 ms at HBM-scale)
#define TDDE_MMA_SHAPES(X) X(5, 1, 1, 6) X(7, 1, 1, 6) X(7, 1, 1, 9)

bool apply_mma_available(int T, int m0, int mstep, int W) {
#define X(t, a, b, w) if (T == t && m0 == a && mstep == b && W == w) return true;
  TDDE_MMA_SHAPES(X)
#undef X
  return false;
}

template <int W>
static void build_frags_w(int T, int n_rad, const std::complex<double>* Rall, std::vector<double>& out) {
  using G = MmaGrid<W>;
  constexpr int ND = 2 * W + 1;
  const int ntile = (n_rad + 7) / 8;
  const int nQ = 2 * (ntile - 1) + G::C0 + 1;
  const int nper = (nQ + 1) / 2;
  const size_t per = (size_t)T * (G::NTL(0) + G::NTL(1)) * 96;
  out.assign(per * nper, 0.0);
  for (int Q = 0; Q < 2 * nper; ++Q) {
    const int par = Q & 1, u = Q >> 1;
    double* base = out.data() + per * u + (par ? (size_t)T * G::NTL(0) * 96 : 0);
    for (int L = 0; L < T; ++L)
      for (int k = 0; k < G::NTL(par); ++k) {
        const int tile = u + G::F(par) + k;
        double* f = base + ((size_t)L * G::NTL(par) + k) * 96;
        for (int lane = 0; lane < 32; ++lane) {
          const int i = 8 * tile + lane / 4, j = 4 * Q - G::OFF + lane % 4;
          if (i < 0 || i >= n_rad || j < 0 || j >= n_rad || i - j > W || j - i > W) continue;
          // column band: Rall[j][L][e] = R_L[j - W + e][j]
          const std::complex<double> c = Rall[((size_t)j * T + L) * ND + (i - j + W)];
          f[lane] = c.real() + c.imag();
          f[32 + lane] = c.real();
          f[64 + lane] = c.imag();
        }
      }
  }
}

// B-operand fragments of every slice (see k_apply_mma) from the column bands Rall[n_rad][T][2W+1]
bool build_mma_frags(int T, int W, int n_rad, const void* Rall, std::vector<double>& out) {
  const std::complex<double>* R = static_cast<const std::complex<double>*>(Rall);
  switch (W) {
    case 3: build_frags_w<3>(T, n_rad, R, out); return true;
    case 6: build_frags_w<6>(T, n_rad, R, out); return true;
    case 9: build_frags_w<9>(T, n_rad, R, out); return true;
    default: return false;
  }
}

int apply_mma_channels(int W) { return mm_nc(W); }

int apply_mma_halo(int W) {     // input rows a segment reads beyond its own, both ends together (for the segment-length choice)
  switch (W) {
    case 3: return 2 * MmaGrid<3>::OFF + 4;
    case 6: return 2 * MmaGrid<6>::OFF + 4;
    case 9: return 2 * MmaGrid<9>::OFF + 4;
    default: return 2 * W + 4;
  }
}

template <int T, int M0, int MS, int W, bool GATHER>
static int launch_mma_one(const ApplyArgs& a, dim3 grid, cudaStream_t s) {
  static bool attr_set[64] = {};
  const size_t smem = MmaPlan<T, M0, MS, W>::SMEM;
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || !attr_set[dev]) {
    if (cudaFuncSetAttribute(k_apply_mma<T, M0, MS, W, GATHER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
    if (dev >= 0 && dev < 64) attr_set[dev] = true;
  }
  k_apply_mma<T, M0, MS, W, GATHER><<<grid, 4 * mm_nc(W), smem, s>>>(a);
  return 1;
}

// y = addv + (coupling terms) x with fused <aux, y>, ||y||^2; a.seg_len must be a multiple of 8
int launch_apply_mma(const ApplyArgs& a, int T, int m0, int mstep, int W, cudaStream_t s) {
  if (!a.addv || !a.Rfrag || (a.emode != 0 && a.emode != 3) || (a.emode == 3 && (!a.aux || !a.y2)) || (a.seg_len & 7)) return -1;
  const int nc = mm_nc(W);
  dim3 grid((a.ld + nc - 1) / nc, (a.n_rad + a.seg_len - 1) / a.seg_len);
#define X(t, aa, b, w)                                                 \
  if (T == t && m0 == aa && mstep == b && W == w)                      \
    return (a.xL || a.xR) ? launch_mma_one<t, aa, b, w, true>(a, grid, s) : launch_mma_one<t, aa, b, w, false>(a, grid, s);
  TDDE_MMA_SHAPES(X)
#undef X
  return -1;
}

// ---- host self-test of the operand table and the slice / tile arithmetic (no GPU): replays what k_apply_mma does with the fragments
// -- slice rows 4Q - OFF + (lane % 4), tiles Q/2 + F(par) + k, B[k][n] = lane 4 n + k, the three Gauss products -- for one channel and
// random z_L, and compares with the band product y[i] = sum_L sum_j R_L[i][j] z_L[j] taken straight from the column bands. ----
template <int W>
static double selftest_frags_w(int T, int n_rad, const std::vector<std::complex<double>>& Rall, const std::vector<std::complex<double>>& z) {
  using G = MmaGrid<W>;
  constexpr int ND = 2 * W + 1;
  std::vector<double> fr;
  build_frags_w<W>(T, n_rad, Rall.data(), fr);
  const int ntile = (n_rad + 7) / 8, nQ = 2 * (ntile - 1) + G::C0 + 1;
  const size_t per = (size_t)T * (G::NTL(0) + G::NTL(1)) * 96;
  std::vector<double> A1((size_t)ntile * 8, 0.0), A2(A1), A3(A1);
  for (int Q = 0; Q < nQ; ++Q) {
    const int par = Q & 1, u = Q >> 1;
    const double* base = fr.data() + per * u + (par ? (size_t)T * G::NTL(0) * 96 : 0);
    for (int L = 0; L < T; ++L)
      for (int k = 0; k < G::NTL(par); ++k) {
        const int tile = u + G::F(par) + k;
        if (tile < 0 || tile >= ntile) continue;
        const double* f = base + ((size_t)L * G::NTL(par) + k) * 96;
        for (int n = 0; n < 8; ++n)
          for (int kk = 0; kk < 4; ++kk) {
            const int j = 4 * Q - G::OFF + kk;
            const std::complex<double> zz = (j >= 0 && j < n_rad) ? z[(size_t)L * n_rad + j] : std::complex<double>(0, 0);
            const int lane = 4 * n + kk;
            A1[(size_t)tile * 8 + n] += zz.real() * f[lane];
            A2[(size_t)tile * 8 + n] += (zz.imag() - zz.real()) * f[32 + lane];
            A3[(size_t)tile * 8 + n] += (zz.real() + zz.imag()) * f[64 + lane];
          }
      }
  }
  double err = 0, nrm = 0;
  for (int i = 0; i < n_rad; ++i) {
    std::complex<double> ref(0, 0);
    for (int L = 0; L < T; ++L)
      for (int j = std::max(0, i - W); j <= std::min(n_rad - 1, i + W); ++j) ref += Rall[((size_t)j * T + L) * ND + (i - j + W)] * z[(size_t)L * n_rad + j];
    const std::complex<double> got(A1[i] - A3[i], A1[i] + A2[i]);
    err = std::max(err, std::abs(got - ref));
    nrm = std::max(nrm, std::abs(ref));
  }
  return nrm > 0 ? err / nrm : err;
}

#ifdef TDDE_WITH_BENCH
extern "C" int tdde_selftest_mma_frags(int32_t n_rad, int32_t w, int32_t T, uint32_t seed, double* max_rel_err) {
  if (n_rad < 1 || T < 1 || !max_rel_err) return TDDE_EINVAL;
  const int ND = 2 * w + 1;
  std::vector<std::complex<double>> Rall((size_t)n_rad * T * ND), z((size_t)T * n_rad);
  uint64_t s = seed * 2654435761u + 12345u;
  auto rnd = [&]() { s = s * 6364136223846793005ull + 1442695040888963407ull; return (double)((s >> 11) & 0xFFFFFFFFu) / 4294967296.0 - 0.5; };
  for (auto& v : Rall) v = {rnd(), rnd()};
  for (auto& v : z) v = {rnd(), rnd()};
  // entries of a column band that point outside the matrix must not matter: poison them
  for (int j = 0; j < n_rad; ++j)
    for (int L = 0; L < T; ++L)
      for (int e = 0; e < ND; ++e) { const int i = j - w + e; if (i < 0 || i >= n_rad) Rall[((size_t)j * T + L) * ND + e] = {1e30, -1e30}; }
  switch (w) {
    case 3: *max_rel_err = selftest_frags_w<3>(T, n_rad, Rall, z); return 0;
    case 6: *max_rel_err = selftest_frags_w<6>(T, n_rad, Rall, z); return 0;
    case 9: *max_rel_err = selftest_frags_w<9>(T, n_rad, Rall, z); return 0;
    default: return TDDE_EINVAL;
  }
}
#endif
