// tdde_eigen.cu -- field-free eigenstates on the device (Eq. 19-20):
//
//     (h0 + kappa h1 + kappa^2 h2 + kappa^3 h3) Psi_kappa = E (s0 + kappa s1 + kappa^2 s2) Psi_kappa ,
//
// one Hermitian-definite pencil (H0_k, S_k) of size n_rad per kappa-class ("2 kappa_max separate eigenvalue problems of
// dimension 2N x 2N"), all eigenpairs, batched over the classes.  Set-up work, not on the time-stepping path: written for
// correctness and simplicity at the sizes the paper uses for it (n_rad of a few hundred).
//   1. S_k = L L^H         banded Cholesky (S_k is banded with half-width w, so L is)
//   2. C = L^-1 H0_k L^-H  two banded forward substitutions on dense columns; C is dense Hermitian
//   3. C = Y diag(E) Y^H   cyclic two-sided Jacobi with the round-robin parallel ordering: n/2 disjoint rotations per round,
//                          first all row updates, then all column updates (and Y <- Y J)
//   4. V = L^-H Y          banded back substitution; the columns of V are S-orthonormal: V^H S V = I
// Eigenvalues are sorted ascending on the host.
#include <algorithm>
#include <cmath>
#include <numeric>
#include <vector>
#include "tdde_handle.h"
#include "tdde_reduce.cuh"

namespace {

// dense row-major [k][i][j] from a row band [k][i][d + w]
__global__ void k_band_to_dense(const cplx* __restrict__ band, cplx* __restrict__ dense, int n, int w) {
  const int k = blockIdx.z, i = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const int d = j - i;
  dense[((size_t)k * n + i) * n + j] = (d >= -w && d <= w) ? band[((size_t)k * n + i) * (2 * w + 1) + d + w] : make_double2(0, 0);
}

// In-place banded Cholesky of the lower band of S (dense storage, only |i - j| <= w touched); one CTA per class.
// ok[k] = 0 when a pivot is not positive.
__global__ void k_chol_banded(cplx* __restrict__ S, int n, int w, int* __restrict__ ok) {
  cplx* A = S + (size_t)blockIdx.x * n * n;
  __shared__ double piv;
  for (int j = 0; j < n; ++j) {
    // column j: rows i = j .. min(n-1, j+w), one thread each: A[i][j] -= sum_{k = max(0, i-w, j-w) .. j-1} A[i][k] conj(A[j][k])
    const int i = j + threadIdx.x;
    cplx v = make_double2(0, 0);
    if (threadIdx.x <= w && i < n) {
      v = A[(size_t)i * n + j];
      for (int k = max(0, i - w); k < j; ++k) {
        const cplx a = A[(size_t)i * n + k], b = A[(size_t)j * n + k];
        v.x -= a.x * b.x + a.y * b.y;
        v.y -= a.y * b.x - a.x * b.y;
      }
    }
    if (threadIdx.x == 0) {
      piv = v.x;
      if (!(v.x > 0.0) || !isfinite(v.x)) ok[blockIdx.x] = 0;
    }
    __syncthreads();
    const double d = sqrt(fabs(piv)) + (piv > 0.0 ? 0.0 : 1.0);
    if (threadIdx.x <= w && i < n) A[(size_t)i * n + j] = (threadIdx.x == 0) ? make_double2(d, 0.0) : make_double2(v.x / d, v.y / d);
    __syncthreads();
  }
}

// B <- L^-1 B for dense B [n][n] (row-major), L banded lower (dense storage); one thread per column of B.
__global__ void k_fwd_sub(const cplx* __restrict__ Lall, cplx* __restrict__ Ball, int n, int w) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const cplx* L = Lall + (size_t)blockIdx.y * n * n;
  cplx* B = Ball + (size_t)blockIdx.y * n * n;
  for (int i = 0; i < n; ++i) {
    cplx v = B[(size_t)i * n + c];
    for (int k = max(0, i - w); k < i; ++k) cfms(v, L[(size_t)i * n + k], B[(size_t)k * n + c]);
    const double d = L[(size_t)i * n + i].x;
    B[(size_t)i * n + c] = make_double2(v.x / d, v.y / d);
  }
}
// B <- L^-H B (back substitution with the upper band L^H); one thread per column of B.
__global__ void k_bwd_sub_h(const cplx* __restrict__ Lall, cplx* __restrict__ Ball, int n, int w) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const cplx* L = Lall + (size_t)blockIdx.y * n * n;
  cplx* B = Ball + (size_t)blockIdx.y * n * n;
  for (int i = n - 1; i >= 0; --i) {
    cplx v = B[(size_t)i * n + c];
    for (int k = i + 1; k <= min(n - 1, i + w); ++k) cfms(v, cconj(L[(size_t)k * n + i]), B[(size_t)k * n + c]);   // (L^H)[i][k] = conj(L[k][i])
    const double d = L[(size_t)i * n + i].x;
    B[(size_t)i * n + c] = make_double2(v.x / d, v.y / d);
  }
}
// out = in^H (dense, per class)
__global__ void k_conj_transpose(const cplx* __restrict__ in, cplx* __restrict__ out, int n) {
  const int k = blockIdx.z, i = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  out[((size_t)k * n + i) * n + j] = cconj(in[((size_t)k * n + j) * n + i]);
}
__global__ void k_identity(cplx* __restrict__ Y, int n) {
  const int k = blockIdx.z, i = blockIdx.y, j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  Y[((size_t)k * n + i) * n + j] = make_double2(i == j ? 1.0 : 0.0, 0.0);
}

// round-robin pairing of m = n rounded up to even players: round r, slot s -> (p, q); an index >= n is a bye
__device__ __forceinline__ void rr_pair(int m, int r, int s, int& p, int& q) {
  const int a = (s == 0) ? m - 1 : (r + s) % (m - 1);
  const int b = (r + m - 1 - s) % (m - 1);
  p = min(a, b); q = max(a, b);
}

// rotation of pair (p, q): J = [[c, s], [-s e^{-i phi}, c e^{-i phi}]] with J^H [[a, b], [conj b, g]] J diagonal
struct Rot { double c, s; cplx e; int p, q; };   // e = e^{i phi}

__global__ void k_jacobi_params(const cplx* __restrict__ Call, Rot* __restrict__ rot, int n, int m, int round) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= m / 2) return;
  const cplx* C = Call + (size_t)blockIdx.y * n * n;
  Rot r;
  rr_pair(m, round, s, r.p, r.q);
  r.c = 1.0; r.s = 0.0; r.e = make_double2(1.0, 0.0);
  if (r.q < n) {
    const double a = C[(size_t)r.p * n + r.p].x, g = C[(size_t)r.q * n + r.q].x;
    const cplx b = C[(size_t)r.p * n + r.q];
    const double ab = hypot(b.x, b.y);
    if (ab > 1e-300 * (fabs(a) + fabs(g)) && ab > 0.0) {
      const double tau = (g - a) / (2.0 * ab);
      const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
      r.c = 1.0 / sqrt(1.0 + t * t);
      r.s = t * r.c;
      r.e = make_double2(b.x / ab, b.y / ab);
    }
  }
  rot[(size_t)blockIdx.y * (m / 2) + s] = r;
}
// rows p, q of C <- J^H (rows):  row_p' = c row_p - s e^{+i phi} row_q ;  row_q' = s row_p + c e^{+i phi} row_q
__global__ void k_jacobi_rows(cplx* __restrict__ Call, const Rot* __restrict__ rot, int n, int m) {
  const Rot r = rot[(size_t)blockIdx.z * (m / 2) + blockIdx.y];
  if (r.q >= n || r.s == 0.0) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  cplx* C = Call + (size_t)blockIdx.z * n * n;
  const cplx xp = C[(size_t)r.p * n + j], xq = C[(size_t)r.q * n + j];
  const cplx eq = cmul(r.e, xq);
  C[(size_t)r.p * n + j] = make_double2(r.c * xp.x - r.s * eq.x, r.c * xp.y - r.s * eq.y);
  C[(size_t)r.q * n + j] = make_double2(r.s * xp.x + r.c * eq.x, r.s * xp.y + r.c * eq.y);
}
// columns p, q of C and of Y <- (cols) J:  col_p' = c col_p - s e^{-i phi} col_q ;  col_q' = s col_p + c e^{-i phi} col_q
__global__ void k_jacobi_cols(cplx* __restrict__ Call, cplx* __restrict__ Yall, const Rot* __restrict__ rot, int n, int m) {
  const Rot r = rot[(size_t)blockIdx.z * (m / 2) + blockIdx.y];
  if (r.q >= n || r.s == 0.0) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const cplx ec = cconj(r.e);
#pragma unroll
  for (int which = 0; which < 2; ++which) {
    cplx* M = (which == 0 ? Call : Yall) + (size_t)blockIdx.z * n * n;
    const cplx xp = M[(size_t)i * n + r.p], xq = M[(size_t)i * n + r.q];
    const cplx eq = cmul(ec, xq);
    M[(size_t)i * n + r.p] = make_double2(r.c * xp.x - r.s * eq.x, r.c * xp.y - r.s * eq.y);
    M[(size_t)i * n + r.q] = make_double2(r.s * xp.x + r.c * eq.x, r.s * xp.y + r.c * eq.y);
  }
}
// off[k] = sum_{i != j} |C_ij|^2, dia[k] = sum_i |C_ii|^2 (one CTA per class; convergence test, read by the host once per sweep)
__global__ void __launch_bounds__(256) k_off_norm(const cplx* __restrict__ Call, double* __restrict__ off, double* __restrict__ dia, int n) {
  const cplx* C = Call + (size_t)blockIdx.x * n * n;
  double o = 0, d = 0;
  for (size_t q = threadIdx.x; q < (size_t)n * n; q += 256) {
    const cplx v = C[q];
    const double m2 = v.x * v.x + v.y * v.y;
    if (q / n == q % n) d += m2; else o += m2;
  }
  __shared__ double so[256], sd[256];
  so[threadIdx.x] = o; sd[threadIdx.x] = d;
  __syncthreads();
  for (int st = 128; st > 0; st >>= 1) {
    if (threadIdx.x < st) { so[threadIdx.x] += so[threadIdx.x + st]; sd[threadIdx.x] += sd[threadIdx.x + st]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { off[blockIdx.x] = so[0]; dia[blockIdx.x] = sd[0]; }
}

}  // namespace

extern "C" int tdde_eigensolve(int32_t n_cls, int32_t n_rad, int32_t w0, const tdde_c64* S_band, const tdde_c64* H0_band, double* E_host,
                               tdde_c64* V_host, void* cuda_stream) {
  if (n_cls <= 0 || n_rad <= 1 || n_rad > 4096 || w0 < 1 || w0 >= n_rad || !S_band || !H0_band || !E_host) return TDDE_EINVAL;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev));
  if (ndev <= 0) { g_last_cuda_error = "no CUDA device"; return TDDE_ECUDA; }
  const int n = n_rad, nd = 2 * w0 + 1, m = (n + 1) / 2 * 2;
  const size_t dense = (size_t)n_cls * n * n, band = (size_t)n_cls * n * nd;
  cplx *dS = nullptr, *dH = nullptr, *dY = nullptr, *dB = nullptr;
  Rot* dR = nullptr;
  int* dOk = nullptr;
  double* dN = nullptr;
  auto cleanup = [&]() { cudaFree(dS); cudaFree(dH); cudaFree(dY); cudaFree(dB); cudaFree(dR); cudaFree(dOk); cudaFree(dN); };
  int rc = 0;
#define EG(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = tdde_cuda_fail(e__, #call); cleanup(); return rc; } } while (0)
  EG(cudaMalloc((void**)&dS, dense * sizeof(cplx)));
  EG(cudaMalloc((void**)&dH, dense * sizeof(cplx)));
  EG(cudaMalloc((void**)&dY, dense * sizeof(cplx)));
  EG(cudaMalloc((void**)&dB, band * sizeof(cplx)));
  EG(cudaMalloc((void**)&dR, (size_t)n_cls * (m / 2) * sizeof(Rot)));
  EG(cudaMalloc((void**)&dOk, n_cls * sizeof(int)));
  EG(cudaMalloc((void**)&dN, 2 * n_cls * sizeof(double)));
  const dim3 ge((n + 127) / 128, n, n_cls);
  EG(cudaMemcpyAsync(dB, S_band, band * sizeof(cplx), cudaMemcpyHostToDevice, s));
  k_band_to_dense<<<ge, 128, 0, s>>>(dB, dS, n, w0);
  EG(cudaMemcpyAsync(dB, H0_band, band * sizeof(cplx), cudaMemcpyHostToDevice, s));
  k_band_to_dense<<<ge, 128, 0, s>>>(dB, dH, n, w0);
  {
    std::vector<int> ones(n_cls, 1);
    EG(cudaMemcpyAsync(dOk, ones.data(), n_cls * sizeof(int), cudaMemcpyHostToDevice, s));
    EG(cudaStreamSynchronize(s));
  }
  // 1. S = L L^H
  k_chol_banded<<<n_cls, 64, 0, s>>>(dS, n, w0, dOk);
  // 2. C = L^-1 H L^-H:  H <- L^-1 H ;  Y <- H^H ;  Y <- L^-1 Y (= L^-1 H^H L^-H ... = C^H = C) ; H <- Y^H
  const dim3 gc((n + 127) / 128, n_cls);
  k_fwd_sub<<<gc, 128, 0, s>>>(dS, dH, n, w0);
  k_conj_transpose<<<ge, 128, 0, s>>>(dH, dY, n);
  k_fwd_sub<<<gc, 128, 0, s>>>(dS, dY, n, w0);
  k_conj_transpose<<<ge, 128, 0, s>>>(dY, dH, n);
  k_identity<<<ge, 128, 0, s>>>(dY, n);
  {
    std::vector<int> ok(n_cls);
    EG(cudaMemcpyAsync(ok.data(), dOk, n_cls * sizeof(int), cudaMemcpyDeviceToHost, s));
    EG(cudaStreamSynchronize(s));
    for (int k = 0; k < n_cls; ++k)
      if (!ok[k]) { cleanup(); return TDDE_ESINGULAR; }     // S_k is not positive definite
  }
  // 3. cyclic Jacobi sweeps until the off-diagonal weight is at rounding level
  std::vector<double> nrm(2 * n_cls);
  const dim3 gp((m / 2 + 63) / 64, n_cls), gr((n + 127) / 128, m / 2, n_cls);
  for (int sweep = 0; sweep < 30; ++sweep) {
    for (int r = 0; r < m - 1; ++r) {
      k_jacobi_params<<<gp, 64, 0, s>>>(dH, dR, n, m, r);
      k_jacobi_rows<<<gr, 128, 0, s>>>(dH, dR, n, m);
      k_jacobi_cols<<<gr, 128, 0, s>>>(dH, dY, dR, n, m);
    }
    k_off_norm<<<n_cls, 256, 0, s>>>(dH, dN, dN + n_cls, n);
    EG(cudaMemcpyAsync(nrm.data(), dN, 2 * n_cls * sizeof(double), cudaMemcpyDeviceToHost, s));
    EG(cudaStreamSynchronize(s));
    bool done = true;
    for (int k = 0; k < n_cls; ++k) done = done && (nrm[k] <= 1e-30 * nrm[n_cls + k]);
    if (done) break;
  }
  // 4. V = L^-H Y
  k_bwd_sub_h<<<gc, 128, 0, s>>>(dS, dY, n, w0);
  EG(cudaGetLastError());
  // eigenvalues = diag(C); sort ascending on the host and hand the eigenvectors over as rows
  std::vector<zc> C(dense), Y(V_host ? dense : 0);
  EG(cudaMemcpyAsync(C.data(), dH, dense * sizeof(cplx), cudaMemcpyDeviceToHost, s));
  if (V_host) EG(cudaMemcpyAsync(Y.data(), dY, dense * sizeof(cplx), cudaMemcpyDeviceToHost, s));
  EG(cudaStreamSynchronize(s));
  zc* Vh = reinterpret_cast<zc*>(V_host);
  std::vector<int> perm(n);
  for (int k = 0; k < n_cls; ++k) {
    const zc* Ck = C.data() + (size_t)k * n * n;
    std::iota(perm.begin(), perm.end(), 0);
    std::sort(perm.begin(), perm.end(), [&](int a, int b) { return Ck[(size_t)a * n + a].real() < Ck[(size_t)b * n + b].real(); });
    for (int e = 0; e < n; ++e) {
      E_host[(size_t)k * n + e] = Ck[(size_t)perm[e] * n + perm[e]].real();
      if (Vh)
        for (int j = 0; j < n; ++j) Vh[((size_t)k * n + e) * n + j] = Y[((size_t)k * n + j) * n + perm[e]];
    }
  }
  cleanup();
#undef EG
  return 0;
}
