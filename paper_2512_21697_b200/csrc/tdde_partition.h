// tdde_partition.h -- host-side set-up of the partitioned (substructured) banded solve used by the preconditioner.
//
// M_k = S_k + i dt/2 H0_k (Eq. 26) is banded with half-width w along r.  A triangular solve is a serial
// recurrence of length n_rad and there are only N_ang independent channels, far too few to fill 148 SMs.  So the
// radial index is cut into P interiors I_0..I_{P-1} separated by P-1 separators of w consecutive rows.  Removing
// the separators decouples the interiors exactly (band half-width w), hence with x = (x_I, x_S):
//     t_I = A_II^{-1} b_I                       P independent banded LU solves per channel        (kernel A)
//     Sc x_S = b_S - A_SI t_I,  Sc = A_SS - A_SI E,  E = A_II^{-1} A_IS   (dense, (P-1) w unknowns) (kernel B)
//     x_I = t_I - E x_S                          2 w complex FMAs per row, fully parallel           (kernel C)
// This is an exact reordering of Gaussian elimination (no truncation).  E ("spikes"), Sc^{-1} and the separator
// rows of M are precomputed here per kappa-class.  Interior blocks are principal submatrices of M_k, whose
// Hermitian part is a principal submatrix of S_k > 0, so LU without pivoting stays safe for them.
#pragma once
#include <complex>
#include <vector>

typedef std::complex<double> zc;

struct PartitionPlan {
  int P = 1;                  // number of interiors
  int w = 0, n = 0;
  std::vector<int> lo, hi;    // interior q = rows [lo[q], hi[q]); separator after it = rows [hi[q], lo[q+1])
  int ns() const { return (P - 1) * w; }
};

PartitionPlan make_partition_plan(int n, int w, int P);

// Mrow: row-band [n][2w+1] of one class, entries pointing outside the matrix already zeroed.
// Outputs (caller-sized): Lcol [n][w], Ucol [n][w+1] (layout of tdde_precond.cu; separator rows = identity),
// Esp [n][2w] (E^- then E^+ per interior row, zero on separator rows), Msep [ns][2w+1] (separator rows of M with
// the separator's own columns zeroed), Scinv [ns][ns].  Returns false on a zero pivot.
bool build_partitioned_factors(const std::vector<zc>& Mrow, const PartitionPlan& plan, zc* Lcol, zc* Ucol, zc* Esp,
                               zc* Msep, zc* Scinv);
