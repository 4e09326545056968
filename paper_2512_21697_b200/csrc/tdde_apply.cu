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
#include "tdde_reduce.cuh"

#define AP_NT 128

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

template <int T, int M0, int MS, int W>
__global__ void __launch_bounds__(AP_NT) k_apply_banded(const ApplyArgs p) {
  using SH = BandShape<T, M0, MS>;
  constexpr int ND = 2 * W + 1;
  constexpr int MAXM = SH::maxm();
  constexpr int NS = SH::nslots();
  if (p.guard == 1 && solver_idle(p.red.st)) return;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;

  const int a = blockIdx.x * AP_NT + threadIdx.x;         // channel (may be a pad lane: a < ld always)
  const int ld = p.ld, n_rad = p.n_rad;
  const bool lane_ok = a < ld;
  const int ac = lane_ok ? a : ld - 1;
  const int i0 = blockIdx.y * p.seg_len;
  const int i1 = min(n_rad, i0 + p.seg_len);

  // angular coefficients in registers, pre-multiplied by beta * g_L
  cplx Areg[NS > 0 ? NS : 1];
  if (T > 0) {
    const double* g = p.g + (p.step_ptr ? (size_t)(*p.step_ptr) * T : 0);
#pragma unroll
    for (int L = 0; L < T; ++L) {
      const double gl = g[L];
      const cplx coef = make_double2(p.beta.x * gl, p.beta.y * gl);
#pragma unroll
      for (int q = 0; q < 2 * SH::m(L); ++q) {
        const int s = SH::slot0(L) + q;
        Areg[s] = cmul(coef, p.Aoff[(size_t)s * ld + ac]);
      }
    }
  }
  const int k = p.cls[ac];
  const cplx* blk = p.blk + (size_t)k * n_rad * ND;

  cplx yw[ND];
#pragma unroll
  for (int e = 0; e < ND; ++e) yw[e] = make_double2(0, 0);
  cplx d0 = make_double2(0, 0);
  double d1 = 0;

  for (int j = i0 - W; j < i1 + W; ++j) {
    if (j >= 0 && j < n_rad) {
      const cplx* xr = p.x + (size_t)j * ld;
      const cplx x0 = xr[ac];
      // block part: per-lane class coefficients
      const cplx* bc = blk + (size_t)j * ND;
#pragma unroll
      for (int e = 0; e < ND; ++e) cfma(yw[e], __ldg(bc + e), x0);
      if (T > 0) {
        cplx z[T > 0 ? T : 1];
#pragma unroll
        for (int L = 0; L < T; ++L) z[L] = make_double2(0, 0);
#pragma unroll
        for (int o = -MAXM; o <= MAXM; ++o) {
          if (o == 0) continue;
          const int ao = min(max(ac + o, 0), ld - 1);      // clamped: the matching A entry is 0 there
          const cplx xo = xr[ao];
#pragma unroll
          for (int L = 0; L < T; ++L) {
            if (SH::m(L) >= (o < 0 ? -o : o)) {
              // slot order within a term: o = -m..-1 -> q = o + m ; o = 1..m -> q = m + o - 1
              const int q = o < 0 ? o + SH::m(L) : SH::m(L) + o - 1;
              cfma(z[L], Areg[SH::slot0(L) + q], xo);
            }
          }
        }
#pragma unroll
        for (int L = 0; L < T; ++L) {
          const cplx* rc = p.Rcol[L] + (size_t)j * ND;      // warp-uniform address
#pragma unroll
          for (int e = 0; e < ND; ++e) cfma(yw[e], __ldg(rc + e), z[L]);
        }
      }
    }
    // row i = j - W is complete
    const int i = j - W;
    if (i >= i0 && i < i1 && lane_ok) {
      const cplx yv = yw[0];
      p.y[(size_t)i * ld + a] = yv;
      if (p.aux) {
        const cplx ax = p.aux[(size_t)i * ld + a];
        cfma_conj(d0, ax, yv);
      }
      d1 = fma(yv.x, yv.x, d1); d1 = fma(yv.y, yv.y, d1);
    }
#pragma unroll
    for (int e = 0; e < ND - 1; ++e) yw[e] = yw[e + 1];
    yw[ND - 1] = make_double2(0, 0);
  }
  if (p.red.fin != FIN_NONE) grid_reduce_finalize<AP_NT>(d0.x, d0.y, d1, p.red);
}

// ---- generic path: arbitrary CSR A_L, arbitrary per-term bandwidths; one thread per output element. ----
// Correct for any input the ABI accepts (e.g. the selection-rule-sparse hydrogen coupling); not tuned.
__global__ void __launch_bounds__(AP_NT) k_apply_generic(const ApplyArgs p) {
  if (p.guard == 1 && solver_idle(p.red.st)) return;
  if (p.guard == 2 && (p.red.st->stalled | (p.red.st->status != 0))) return;
  const int a = blockIdx.x * AP_NT + threadIdx.x;
  const int i = blockIdx.y;
  const int ld = p.ld, n_rad = p.n_rad;
  cplx d0 = make_double2(0, 0);
  double d1 = 0;
  if (a < ld) {
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
    p.y[(size_t)i * ld + a] = acc;
    if (p.aux) cfma_conj(d0, p.aux[(size_t)i * ld + a], acc);
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

bool apply_banded_available(int T, int m0, int mstep, int W) {
#define X(t, a, b, w) if (T == t && (t == 0 || (m0 == a && mstep == b)) && W == w) return true;
  TDDE_BANDED_SHAPES(X)
#undef X
  return false;
}

int launch_apply_banded(const ApplyArgs& a, int T, int m0, int mstep, int W, cudaStream_t s) {
  dim3 grid((a.ld + AP_NT - 1) / AP_NT, (a.n_rad + a.seg_len - 1) / a.seg_len);
#define X(t, aa, b, w) \
  if (T == t && (t == 0 || (m0 == aa && mstep == b)) && W == w) { k_apply_banded<t, aa, b, w><<<grid, AP_NT, 0, s>>>(a); return 1; }
  TDDE_BANDED_SHAPES(X)
#undef X
  return -1;
}

int launch_apply_generic(const ApplyArgs& a, cudaStream_t s) {
  dim3 grid((a.ld + AP_NT - 1) / AP_NT, a.n_rad);
  k_apply_generic<<<grid, AP_NT, 0, s>>>(a);
  return 1;
}
