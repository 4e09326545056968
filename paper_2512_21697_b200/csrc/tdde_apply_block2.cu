// tdde_apply_block2.cu -- start of a CN step, block parts only: ONE pass over c gives  u = oscale * H0 c  and  v = S c
// (SURVEY 8(a) a2 + a3; R6: b = S c + r0 / 2, r0 = -i dt (H0 c + sum_L g_L (A_L (x) R_L) c)).
// The coupling part of r0 is then added by the DMMA apply (tdde_apply_mma.cu), whose epilogue also forms ||b||^2 and ||r0||^2.
// HBM-bound (16 B read, 32 B written, 2 (2W+1) complex FMAs per element): lane <-> channel, a thread walks a radial segment in
// scatter form with two register windows; the x rows and the column coefficients of the CTA's kappa-classes (both operators) arrive
// by 1-D TMA bulk copies in a three-stage mbarrier ring.
#include "tdde_reduce.cuh"

#define B2_NC TDDE_AP_NC
#ifndef B2_JC
#define B2_JC 4
#endif
#ifndef B2_NST
#define B2_NST 3      // measured: 4 stages lose (HBM-scale step 7.87 -> 8.36 ms)
#endif
#define B2_MAXC TDDE_AP_MAXC
#ifndef B2_RU
#define B2_RU 1
#endif
#ifndef B2_MINB9
#define B2_MINB9 1
#endif
#ifndef B2_MINB6
#define B2_MINB6 2
#endif

namespace {
__device__ __forceinline__ uint32_t b2_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void b2_bar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(b2_smem(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void b2_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b2_smem(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void b2_bulk(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(b2_smem(dst)),
               "l"(src), "r"(bytes), "r"(b2_smem(bar))
               : "memory");
}
__device__ __forceinline__ void b2_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok)
                 : "r"(b2_smem(bar)), "r"(parity)
                 : "memory");
  } while (!ok);
}
}  // namespace

// stage = [blk: ncm classes x JC rows x ND][blk2: same][x: JC rows x 128]; ncm = the largest number of kappa-classes any CTA stages
template <int W>
struct Block2Plan {
  static constexpr int ND = 2 * W + 1;
  __host__ __device__ static int cs(int ncm) { return ncm * B2_JC * ND; }
  __host__ __device__ static int stage(int ncm) { return 2 * cs(ncm) + B2_JC * B2_NC; }
  static size_t smem(int ncm) { return (size_t)B2_NST * stage(ncm) * sizeof(cplx) + 64; }
};

// p.x -> p.y = oscale * (blk) x, p.y2 = (blk2) x; blk / blk2 in column-band form [n_cls][n_rad][2W+1]
template <int W>
__global__ void __launch_bounds__(2 * B2_NC, (W <= 3 ? 4 : W <= 6 ? B2_MINB6 : B2_MINB9)) k_block_dual(const __grid_constant__ ApplyArgs p, const cplx* __restrict__ blk2) {
  using PL = Block2Plan<W>;
  constexpr int ND = PL::ND, JC = B2_JC, RU = B2_RU;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  cplx* stage_base = reinterpret_cast<cplx*>(smem_raw);
  const int CS = PL::cs(p.n_cta_cls), STAGE = PL::stage(p.n_cta_cls);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)B2_NST * STAGE * sizeof(cplx));

  // 256 threads: threads [0, 128) form (blk) x, threads [128, 256) form (blk2) x from the same staged x rows -- one 2W+1 window per
  // thread instead of two (half the registers, twice the warps per SM)
  const int tid = threadIdx.x % B2_NC, op = threadIdx.x / B2_NC, ld = p.ld, n_rad = p.n_rad;
  const cplx* const blk_g = op ? blk2 : p.blk;
  const int a0 = blockIdx.x * B2_NC, a = a0 + tid;
  const bool lane_ok = a >= p.own_lo && a < p.own_hi;          // own_hi <= ld
  const int ac = a < ld ? a : ld - 1;
  const int i0 = blockIdx.y * p.seg_len, i1 = min(n_rad, i0 + p.seg_len);
  const int jlo = max(0, i0 - W), jhi = min(n_rad, i1 + W), jend = i1 + W;
  const int nchunks = (jend - jlo + JC - 1) / JC;
  const int slot = p.slot[ac] < p.n_cta_cls ? p.slot[ac] : -1;   // classes beyond the staged ones: coefficients from global (L1 / L2)
  const size_t cls_off = (size_t)p.cls[ac] * n_rad * ND;
  const int* cta_cls = p.cta_cls + blockIdx.x * B2_MAXC;
  const int nch = min(B2_NC, ld - a0);                        // channels of this CTA inside the vector
  if (nch < B2_NC)
    for (int q = threadIdx.x; q < B2_NST * STAGE; q += 2 * B2_NC) stage_base[q] = make_double2(0, 0);
  if (threadIdx.x == 0) {
    for (int q = 0; q < B2_NST; ++q) b2_bar_init(&full[q], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");

  auto issue = [&](int c) {
    cplx* st = stage_base + (size_t)(c % B2_NST) * STAGE;
    uint64_t* bar = &full[c % B2_NST];
    const int j = jlo + c * JC;
    const int nr = min(JC, jhi - j);
    if (nr <= 0) return;
    int ncls = 0;
#pragma unroll
    for (int q = 0; q < B2_MAXC; ++q) ncls += (q < p.n_cta_cls && cta_cls[q] >= 0);
    const bool x2d = p.use_xmap != 0;                           // one tensor copy for the x rows: full box, out-of-bounds zero-filled
    b2_expect_tx(bar, (uint32_t)((2 * ncls * nr * ND + (x2d ? JC * B2_NC : nr * nch)) * sizeof(cplx)));
#pragma unroll
    for (int q = 0; q < B2_MAXC; ++q) {
      const int kk = q < p.n_cta_cls ? cta_cls[q] : -1;
      if (kk >= 0) {
        b2_bulk(st + (size_t)q * JC * ND, p.blk + ((size_t)kk * n_rad + j) * ND, (uint32_t)nr * ND * sizeof(cplx), bar);
        b2_bulk(st + CS + (size_t)q * JC * ND, blk2 + ((size_t)kk * n_rad + j) * ND, (uint32_t)nr * ND * sizeof(cplx), bar);
      }
    }
    if (x2d) {
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                       b2_smem(st + 2 * CS)),
                   "l"(reinterpret_cast<uint64_t>(&p.xmap)), "r"(2 * a0), "r"(j), "r"(b2_smem(bar))
                   : "memory");
    } else {
      for (int r = 0; r < nr; ++r)
        b2_bulk(st + 2 * CS + (size_t)r * B2_NC, p.x + (size_t)(j + r) * ld + a0, (uint32_t)nch * sizeof(cplx), bar);
    }
  };
  if (threadIdx.x == 0)
    for (int c = 0; c < B2_NST && c < nchunks; ++c) issue(c);

  cplx w1[ND];
#pragma unroll
  for (int e = 0; e < ND; ++e) w1[e] = make_double2(0, 0);
  for (int c = 0; c < nchunks; ++c) {
    const cplx* st = stage_base + (size_t)(c % B2_NST) * STAGE;
    const int jc0 = jlo + c * JC;
    const int nr_real = min(JC, jhi - jc0), nr_all = min(JC, jend - jc0);
    if (nr_real > 0) b2_wait(&full[c % B2_NST], (c / B2_NST) & 1);
#pragma unroll(RU)
    for (int r = 0; r < JC; ++r) {
      if (r < nr_all) {
        if (r < nr_real) {
          const cplx x0 = st[2 * CS + r * B2_NC + tid];
          if (slot >= 0) {
            const cplx* c1 = st + (size_t)op * CS + ((size_t)slot * JC + r) * ND;
#pragma unroll
            for (int e = 0; e < ND; ++e) cfma(w1[e], c1[e], x0);
          } else {
            const cplx* c1 = blk_g + cls_off + (size_t)(jc0 + r) * ND;
#pragma unroll
            for (int e = 0; e < ND; ++e) cfma(w1[e], __ldg(c1 + e), x0);
          }
        }
        const int i = jc0 + r - W;
        if (i >= i0 && lane_ok) {
          if (op == 0) p.y[(size_t)i * ld + a] = cmul(p.oscale, w1[0]);
          else p.y2[(size_t)i * ld + a] = w1[0];
        }
#pragma unroll
        for (int e = 0; e < ND - 1; ++e) w1[e] = w1[e + 1];
        w1[ND - 1] = make_double2(0, 0);
      }
    }
    __syncthreads();                                            // everybody is done with stage c % NST
    if (threadIdx.x == 0 && c + B2_NST < nchunks) issue(c + B2_NST);
  }
}

template <int W>
static int launch_block_dual_w(const ApplyArgs& a, const cplx* blk2, cudaStream_t s) {
  static bool attr_set[64] = {};
  const size_t smem = Block2Plan<W>::smem(a.n_cta_cls);
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64 || !attr_set[dev]) {
    if (cudaFuncSetAttribute(k_block_dual<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Block2Plan<W>::smem(B2_MAXC)) != cudaSuccess) return -2;
    if (dev >= 0 && dev < 64) attr_set[dev] = true;
  }
  dim3 grid((a.ld + B2_NC - 1) / B2_NC, (a.n_rad + a.seg_len - 1) / a.seg_len);
  k_block_dual<W><<<grid, 2 * B2_NC, smem, s>>>(a, blk2);
  return 1;
}

// y = oscale * (blk) x, y2 = (blk2) x; W = the (padded) half-bandwidth of the banded path's column bands
int launch_block_dual(const ApplyArgs& a, const cplx* blk2, int W, cudaStream_t s) {
  switch (W) {
    case 3: return launch_block_dual_w<3>(a, blk2, s);
    case 6: return launch_block_dual_w<6>(a, blk2, s);
    case 9: return launch_block_dual_w<9>(a, blk2, s);
    default: return -1;
  }
}
