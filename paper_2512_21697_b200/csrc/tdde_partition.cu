// tdde_partition.cu -- host code (one-time, per kappa-class): see tdde_partition.h.
#include <algorithm>
#include <cmath>
#include "tdde_internal.h"
#include "tdde_partition.h"

static int min_interior(int w) { return std::max(2 * w, 8); }

PartitionPlan make_partition_plan(int n, int w, int P) {
  PartitionPlan pl;
  pl.n = n; pl.w = w;
  P = std::max(1, P);
  while (P > 1 && (n - (P - 1) * w) / P < min_interior(w)) --P;     // block-tridiagonal Schur needs interiors >= w rows
  pl.P = P;
  const int interior = n - (P - 1) * w;
  int pos = 0;
  for (int q = 0; q < P; ++q) {
    const int m = interior / P + (q < interior % P ? 1 : 0);
    pl.lo.push_back(pos);
    pl.hi.push_back(pos + m);
    pos += m + w;
  }
  return pl;
}

int partitions_for_rows(int n, int w, int rows) {
  rows = std::max(rows, min_interior(w));
  return std::max(1, (n + w + rows + w - 1) / (rows + w));
}

namespace {

// segment id of a row: 2q for interior q, 2q+1 for the separator after interior q
int segment_of(const PartitionPlan& pl, int i) {
  for (int q = 0; q < pl.P; ++q) {
    if (i < pl.hi[q]) return 2 * q;
    if (q + 1 < pl.P && i < pl.lo[q + 1]) return 2 * q + 1;
  }
  return 2 * (pl.P - 1);
}

bool invert_dense(std::vector<zc>& A, int n, zc* out) {   // Gauss-Jordan, partial pivoting
  std::vector<zc> I((size_t)n * n, zc(0, 0));
  for (int i = 0; i < n; ++i) I[(size_t)i * n + i] = zc(1, 0);
  for (int c = 0; c < n; ++c) {
    int piv = c;
    double best = std::abs(A[(size_t)c * n + c]);
    for (int r = c + 1; r < n; ++r)
      if (std::abs(A[(size_t)r * n + c]) > best) { best = std::abs(A[(size_t)r * n + c]); piv = r; }
    if (!(best > TDDE_TINY) || !std::isfinite(best)) return false;
    if (piv != c)
      for (int j = 0; j < n; ++j) { std::swap(A[(size_t)c * n + j], A[(size_t)piv * n + j]); std::swap(I[(size_t)c * n + j], I[(size_t)piv * n + j]); }
    const zc inv = zc(1, 0) / A[(size_t)c * n + c];
    for (int j = 0; j < n; ++j) { A[(size_t)c * n + j] *= inv; I[(size_t)c * n + j] *= inv; }
    for (int r = 0; r < n; ++r) {
      if (r == c) continue;
      const zc f = A[(size_t)r * n + c];
      if (f == zc(0, 0)) continue;
      for (int j = 0; j < n; ++j) { A[(size_t)r * n + j] -= f * A[(size_t)c * n + j]; I[(size_t)r * n + j] -= f * I[(size_t)c * n + j]; }
    }
  }
  std::copy(I.begin(), I.end(), out);
  return true;
}

}  // namespace

bool build_partitioned_factors(const std::vector<zc>& Mrow, const PartitionPlan& pl, zc* Lcol, zc* Ucol, zc* Wsp,
                               zc* Corner, zc* Schur, double* growth) {
  const int n = pl.n, w = pl.w, nd = 2 * w + 1, P = pl.P;
  auto M = [&](int i, int j) -> zc { return (j < 0 || j >= n || std::abs(i - j) > w) ? zc(0, 0) : Mrow[(size_t)i * nd + (j - i + w)]; };
  std::vector<int> seg(n);
  for (int i = 0; i < n; ++i) seg[i] = segment_of(pl, i);

  // block-diagonal copy: couplings between different segments removed, separators replaced by identity
  std::vector<zc> F(Mrow);
  double max_m = 0;
  for (int i = 0; i < n; ++i)
    for (int d = -w; d <= w; ++d) {
      const int j = i + d;
      if (j < 0 || j >= n) { F[(size_t)i * nd + d + w] = zc(0, 0); continue; }
      max_m = std::max(max_m, std::abs(F[(size_t)i * nd + d + w]));
      if (seg[i] % 2 == 1) F[(size_t)i * nd + d + w] = (d == 0) ? zc(1, 0) : zc(0, 0);
      else if (seg[j] != seg[i]) F[(size_t)i * nd + d + w] = zc(0, 0);
    }
  auto at = [&](int i, int j) -> zc& { return F[(size_t)i * nd + (j - i + w)]; };
  // LU without pivoting, in place (block-diagonal structure is preserved: no fill across zeroed couplings)
  for (int i = 0; i < n; ++i) {
    const zc piv = at(i, i);
    if (!(std::isfinite(piv.real()) && std::isfinite(piv.imag())) || std::abs(piv) < TDDE_TINY) return false;
    const int last = std::min(i + w, n - 1);
    for (int r = i + 1; r <= last; ++r) {
      if (at(r, i) == zc(0, 0)) continue;
      const zc l = at(r, i) / piv;
      at(r, i) = l;
      for (int c = i + 1; c <= last; ++c) at(r, c) -= l * at(i, c);
    }
  }
  if (growth) {
    double max_lu = 0;
    for (size_t q = 0; q < F.size(); ++q) max_lu = std::max(max_lu, std::abs(F[q]));
    *growth = max_m > 0 ? max_lu / max_m : 1.0;
  }
  for (int i = 0; i < n; ++i) {
    for (int d = 1; d <= w; ++d) Lcol[(size_t)i * w + d - 1] = (i + d < n) ? at(i + d, i) : zc(0, 0);
    const zc uinv = zc(1, 0) / at(i, i);
    Ucol[(size_t)i * (w + 1)] = uinv;
    for (int d = 1; d <= w; ++d) Ucol[(size_t)i * (w + 1) + d] = (i - d >= 0) ? at(i - d, i) : zc(0, 0);
    Ucol[(size_t)i * (w + 1) + 1] *= uinv;     // pre-scaled: shortens the dependent chain of the U sweep
  }
  if (P == 1) return true;

  // left spikes: row s of W = A_SI A_II^{-1} restricted to interior q solves A_qq^T u = M[s, I_q]^T; with A_qq = L U
  // that is U^T z = a (forward), L^T u = z (backward)
  std::fill(Wsp, Wsp + (size_t)n * 2 * w, zc(0, 0));
  std::vector<zc> z(n), u(n);
  for (int q = 0; q < P; ++q) {
    const int lo = pl.lo[q], hi = pl.hi[q];
    for (int side = 0; side < 2; ++side) {
      if ((side == 0 && q == 0) || (side == 1 && q == P - 1)) continue;
      const int s0 = side == 0 ? pl.hi[q - 1] : pl.hi[q];
      for (int c = 0; c < w; ++c) {
        const int s = s0 + c;
        for (int i = lo; i < hi; ++i) {
          zc acc = M(s, i);
          for (int d = 1; d <= w && i - d >= lo; ++d) acc -= at(i - d, i) * z[i - d];
          z[i] = acc / at(i, i);
        }
        for (int i = hi - 1; i >= lo; --i) {
          zc acc = z[i];
          for (int d = 1; d <= w && i + d < hi; ++d) acc -= at(i + d, i) * u[i + d];
          u[i] = acc;
          Wsp[(size_t)i * 2 * w + side * w + c] = acc;
        }
      }
    }
  }
  // corners of A_IS: the only rows of an interior that see a separator are its first and last w rows
  const size_t ww = (size_t)w * w;
  std::fill(Corner, Corner + (size_t)P * 2 * ww, zc(0, 0));
  for (int q = 0; q < P; ++q)
    for (int r = 0; r < w; ++r)
      for (int c = 0; c < w; ++c) {
        if (q > 0) Corner[((size_t)q * 2 + 0) * ww + r * w + c] = M(pl.lo[q] + r, pl.hi[q - 1] + c);
        if (q + 1 < P) Corner[((size_t)q * 2 + 1) * ww + r * w + c] = M(pl.hi[q] - w + r, pl.hi[q] + c);
      }
  // Schur complement Sc = A_SS - W A_IS, block tridiagonal; block Thomas factors
  std::vector<zc> D(ww), B(ww), C(ww), Cprev(ww, zc(0, 0)), Dinv_prev(ww, zc(0, 0)), Lb(ww), tmp(ww);
  std::fill(Schur, Schur + (size_t)(P - 1) * 3 * ww, zc(0, 0));
  for (int j = 0; j + 1 < P; ++j) {
    const int s0 = pl.hi[j];
    std::fill(B.begin(), B.end(), zc(0, 0));
    std::fill(C.begin(), C.end(), zc(0, 0));
    for (int c = 0; c < w; ++c)
      for (int c2 = 0; c2 < w; ++c2) {
        zc d = M(s0 + c, s0 + c2), b(0, 0), cc(0, 0);
        for (int i = std::max(pl.lo[j], pl.hi[j] - w); i < pl.hi[j]; ++i) d -= Wsp[(size_t)i * 2 * w + w + c] * M(i, s0 + c2);
        for (int i = pl.lo[j + 1]; i < std::min(pl.hi[j + 1], pl.lo[j + 1] + w); ++i) d -= Wsp[(size_t)i * 2 * w + c] * M(i, s0 + c2);
        if (j > 0)
          for (int i = pl.lo[j]; i < std::min(pl.hi[j], pl.lo[j] + w); ++i) b -= Wsp[(size_t)i * 2 * w + w + c] * M(i, pl.hi[j - 1] + c2);
        if (j + 2 < P)
          for (int i = std::max(pl.lo[j + 1], pl.hi[j + 1] - w); i < pl.hi[j + 1]; ++i) cc -= Wsp[(size_t)i * 2 * w + c] * M(i, pl.hi[j + 1] + c2);
        D[c * w + c2] = d; B[c * w + c2] = b; C[c * w + c2] = cc;
      }
    std::fill(Lb.begin(), Lb.end(), zc(0, 0));
    if (j > 0) {
      for (int a = 0; a < w; ++a)
        for (int b2 = 0; b2 < w; ++b2) {
          zc acc(0, 0);
          for (int k = 0; k < w; ++k) acc += B[a * w + k] * Dinv_prev[k * w + b2];
          Lb[a * w + b2] = acc;
        }
      for (int a = 0; a < w; ++a)
        for (int b2 = 0; b2 < w; ++b2) {
          zc acc(0, 0);
          for (int k = 0; k < w; ++k) acc += Lb[a * w + k] * Cprev[k * w + b2];
          D[a * w + b2] -= acc;
        }
    }
    tmp = D;
    if (!invert_dense(tmp, w, Dinv_prev.data())) return false;
    zc* out = Schur + (size_t)j * 3 * ww;
    std::copy(Lb.begin(), Lb.end(), out);
    std::copy(Dinv_prev.begin(), Dinv_prev.end(), out + ww);
    for (int a = 0; a < w; ++a)                                   // G_j = D'^-1_j C_j: x_j = D'^-1_j r'_j - G_j x_{j+1}
      for (int b2 = 0; b2 < w; ++b2) {
        zc acc(0, 0);
        for (int k = 0; k < w; ++k) acc += Dinv_prev[a * w + k] * C[k * w + b2];
        out[2 * ww + a * w + b2] = acc;
      }
    Cprev = C;
  }
  return true;
}

#ifdef TDDE_WITH_BENCH
// ---- host self-test (no GPU): the partitioned solve, with the device kernels P1/P2/P3 replayed in plain loops on the
// host arrays exactly as laid out for the device; checked by the residual of the original banded system ----
extern "C" int tdde_selftest_partition(int32_t n, int32_t w, int32_t P, uint32_t seed, double* max_rel_err) {
  if (n <= 0 || w < 1 || w >= n || P < 1 || !max_rel_err) return TDDE_EINVAL;
  const int nd = 2 * w + 1;
  uint64_t st = seed * 2654435761ull + 12345;
  auto rnd = [&]() { st = st * 6364136223846793005ull + 1442695040888963407ull; return ((st >> 11) & 0xfffff) / 524288.0 - 1.0; };
  // M = S + i tau H with S SPD-ish (strong diagonal) and H Hermitian: the structure of PAPER.md Eq. 26
  std::vector<zc> Mrow((size_t)n * nd, zc(0, 0));
  for (int i = 0; i < n; ++i)
    for (int d = 0; d <= w; ++d) {
      if (i + d >= n) continue;
      const zc s = d == 0 ? zc(2.0 + 0.1 * rnd(), 0) : zc(0.3 * rnd() / d, 0);
      const zc hh = d == 0 ? zc(rnd(), 0) : zc(rnd(), rnd());
      Mrow[(size_t)i * nd + w + d] = s + zc(0, 0.05) * hh;
      if (d > 0) Mrow[(size_t)(i + d) * nd + w - d] = std::conj(s) + zc(0, 0.05) * std::conj(hh);
    }
  const PartitionPlan pl = make_partition_plan(n, w, P);
  const int Pp = pl.P;
  const size_t ww = (size_t)w * w;
  std::vector<zc> Lc((size_t)n * w), Uc((size_t)n * (w + 1)), Wsp((size_t)n * 2 * w + 1), Corner((size_t)Pp * 2 * ww + 1), Sch((size_t)(Pp - 1) * 3 * ww + 1);
  double growth = 0;
  if (!build_partitioned_factors(Mrow, pl, Lc.data(), Uc.data(), Wsp.data(), Corner.data(), Sch.data(), &growth)) return TDDE_ESINGULAR;
  std::vector<zc> b(n), y(n, zc(0, 0));
  for (int i = 0; i < n; ++i) b[i] = zc(rnd(), rnd());
  std::vector<zc> rsm((size_t)Pp * w, zc(0, 0)), rsp((size_t)Pp * w, zc(0, 0));
  if (Pp > 1) {
    // kernel P1: per interior, the spike dot products for the separator before (minus) and after (plus)
    for (int q = 0; q < Pp; ++q)
      for (int i = pl.lo[q]; i < pl.hi[q]; ++i)
        for (int c = 0; c < w; ++c) {
          rsm[(size_t)q * w + c] += Wsp[(size_t)i * 2 * w + c] * b[i];
          rsp[(size_t)q * w + c] += Wsp[(size_t)i * 2 * w + w + c] * b[i];
        }
    // kernel P2: block Thomas over the separators.  Forward: r'_j = r_j - Lb_j r'_{j-1}, z_j = D'^-1_j r'_j (kept in rsp);
    // backward: x_j = z_j - G_j x_{j+1}
    std::vector<zc> prev(w, zc(0, 0)), cur(w), xn(w, zc(0, 0));
    for (int j = 0; j + 1 < Pp; ++j) {
      const zc* Lb = Sch.data() + (size_t)j * 3 * ww;
      const zc* Di = Lb + ww;
      for (int c = 0; c < w; ++c) {
        zc r = b[pl.hi[j] + c] - rsp[(size_t)j * w + c] - rsm[(size_t)(j + 1) * w + c];
        for (int k = 0; k < w; ++k) r -= Lb[c * w + k] * prev[k];
        cur[c] = r;
      }
      for (int c = 0; c < w; ++c) prev[c] = cur[c];
      for (int c = 0; c < w; ++c) {
        zc z(0, 0);
        for (int k = 0; k < w; ++k) z += Di[c * w + k] * prev[k];
        rsp[(size_t)j * w + c] = z;
      }
    }
    for (int j = Pp - 2; j >= 0; --j) {
      const zc* G = Sch.data() + (size_t)j * 3 * ww + 2 * ww;
      for (int c = 0; c < w; ++c) {
        zc x = rsp[(size_t)j * w + c];
        for (int k = 0; k < w; ++k) x -= G[c * w + k] * xn[k];
        cur[c] = x;
      }
      for (int c = 0; c < w; ++c) xn[c] = y[pl.hi[j] + c] = cur[c];
    }
    // kernel P2b: A_IS x_S for the interiors next to each separator
    for (int j = 0; j + 1 < Pp; ++j)
      for (int c = 0; c < w; ++c) {
        zc ct(0, 0), cb(0, 0);
        for (int k = 0; k < w; ++k) {
          ct += Corner[((size_t)(j + 1) * 2 + 0) * ww + c * w + k] * y[pl.hi[j] + k];
          cb += Corner[((size_t)j * 2 + 1) * ww + c * w + k] * y[pl.hi[j] + k];
        }
        rsm[(size_t)(j + 1) * w + c] = ct;
        rsp[(size_t)j * w + c] = cb;
      }
  }
  // kernel P3: per interior, corner-corrected right-hand side, then forward and backward sweep in column form
  for (int q = 0; q < Pp; ++q) {
    const int lo = pl.lo[q], hi = pl.hi[q], len = hi - lo;
    std::vector<zc> tile(len);
    for (int r = 0; r < len; ++r) tile[r] = b[lo + r];
    if (q > 0)
      for (int r = 0; r < w; ++r) tile[r] -= rsm[(size_t)q * w + r];
    if (q + 1 < Pp)
      for (int r = 0; r < w; ++r) tile[len - w + r] -= rsp[(size_t)q * w + r];
    std::vector<zc> pw(w + 1, zc(0, 0));
    for (int r = 0; r < len; ++r) {
      const int i = lo + r;
      tile[r] += pw[0];
      for (int d = 0; d < w; ++d) pw[d] = pw[d + 1] - Lc[(size_t)i * w + d] * tile[r];
    }
    std::fill(pw.begin(), pw.end(), zc(0, 0));
    for (int r = len - 1; r >= 0; --r) {
      const int i = lo + r;
      const zc t = tile[r] + pw[0];
      const zc xi = t * Uc[(size_t)i * (w + 1)];
      y[i] = xi;
      pw[0] = pw[1] - Uc[(size_t)i * (w + 1) + 1] * t;           // pre-scaled entry multiplies (y_i + pw0)
      for (int d = 1; d < w; ++d) pw[d] = pw[d + 1] - Uc[(size_t)i * (w + 1) + d + 1] * xi;
    }
  }
  double num = 0, den = 0;
  for (int i = 0; i < n; ++i) {
    zc acc(0, 0);
    for (int d = -w; d <= w; ++d)
      if (i + d >= 0 && i + d < n) acc += Mrow[(size_t)i * nd + d + w] * y[i + d];
    num += std::norm(acc - b[i]);
    den += std::norm(b[i]);
  }
  *max_rel_err = std::sqrt(num / den);
  return pl.P;        // the partition count actually used (>= 1)
}
#endif  // TDDE_WITH_BENCH
