// tdde_partition.h -- host-side set-up of the partitioned (substructured) banded solve used by the preconditioner.
//
// M_k = S_k + i dt/2 H0_k (Eq. 26) is banded with half-width w along r.  A triangular solve is a serial
// recurrence of length n_rad and there are only N_ang independent channels, far too few to fill 148 SMs, and a plain
// two-sweep solve reads/writes every element twice.  So the radial index is cut into P interiors I_0..I_{P-1}
// separated by P-1 separators of w consecutive rows, short enough that one (32-channel x interior) tile lives in shared
// memory between its L and U sweeps.  Removing the separators decouples the interiors exactly (band half-width w),
// hence with x = (x_I, x_S):
//     r_S = b_S - W b_I,          W = A_SI A_II^{-1}   ("left spikes": 2 w complex FMAs per interior row, streaming)  (kernel P1)
//     Sc x_S = r_S,               Sc = A_SS - W A_IS   (block tridiagonal, blocks w x w: block Thomas per channel)  (kernel P2)
//     x_I = A_II^{-1} (b_I - A_IS x_S)                 (P independent banded LU solves per channel, in shared memory) (kernel P3)
// This is an exact reordering of Gaussian elimination (no truncation).  W, the block-LU of Sc and the corner blocks of
// A_IS are precomputed here per kappa-class.  Interior blocks are principal submatrices of M_k, whose Hermitian part is
// a principal submatrix of S_k > 0, so LU without pivoting stays safe for them; Sc inherits a positive definite Hermitian
// part as a Schur complement of M_k.
#pragma once
#include <complex>
#include <vector>

typedef std::complex<double> zc;

struct PartitionPlan {
  int P = 1;                  // number of interiors
  int w = 0, n = 0;
  std::vector<int> lo, hi;    // interior q = rows [lo[q], hi[q]); separator after it = rows [hi[q], lo[q+1])
  int nsep() const { return P - 1; }
  int max_interior() const {
    int m = 0;
    for (int q = 0; q < P; ++q) m = hi[q] - lo[q] > m ? hi[q] - lo[q] : m;
    return m;
  }
};

// P interiors of (nearly) equal length; P shrinks until every interior has at least max(2 w, 8) rows.
PartitionPlan make_partition_plan(int n, int w, int P);
// The P that gives interiors of about `rows` rows.
int partitions_for_rows(int n, int w, int rows);

// Per-class factors.  Mrow: row-band [n][2w+1] of one class, entries pointing outside the matrix already zeroed.
// Outputs (caller-sized):
//   Lcol  [n][w], Ucol [n][w+1]   LU of the interiors in the layout of tdde_precond.cu (separator rows = identity)
//   Wsp   [n][2w]                 interior row i of interior q: [c] = W[separator q-1, row c][i], [w+c] = W[separator q, row c][i]
//   Corner[P][2][w][w]            A_IS corners: [q][0][r][c] = M[lo_q + r][hi_{q-1} + c], [q][1][r][c] = M[hi_q - w + r][hi_q + c]
//   Schur [P-1][3][w][w]          block Thomas of Sc: [j][0] = B_j D'_{j-1}^{-1}, [j][1] = D'_j^{-1}, [j][2] = D'_j^{-1} C_j (row-major)
// growth (nullable): max |L_ij|, |U_ij| over the interiors divided by max |M_ij| (element growth of the unpivoted LU).
// Returns false on a zero / non-finite pivot.
bool build_partitioned_factors(const std::vector<zc>& Mrow, const PartitionPlan& plan, zc* Lcol, zc* Ucol, zc* Wsp,
                               zc* Corner, zc* Schur, double* growth);
