"""Container for one TDDE Crank-Nicolson problem in the boundary (C-ABI) layout.

Layout conventions (identical to include/tdde.h):

* state vector ``c[a * n_rad + j]``: channel-major, radial-fastest, complex128;
* a radial band matrix R of half-bandwidth w is stored row-major
  ``band[i, d + w] = R[i, i + d]`` for ``-w <= d <= w`` and 0 where ``i + d`` falls
  outside ``[0, n_rad)``;
* field-free blocks are given per kappa-class: ``S_band[k]``, ``H0_band[k]``,
  channel ``a`` uses class ``cls_of_chan[a]`` (blocks depend
  on kappa only);
* one coupling term is ``g_L(t) * (A_L (x) R_L)`` with A_L in CSR
  (Eq. 17).

Nothing here computes with these arrays beyond format conversion.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, List

import numpy as np


@dataclass
class Term:
    w: int
    R_band: np.ndarray      # [n_rad, 2w+1] complex128
    A_rowptr: np.ndarray    # [n_ang+1] int32
    A_col: np.ndarray       # [nnz] int32
    A_val: np.ndarray       # [nnz] complex128


@dataclass
class Problem:
    name: str
    n_ang: int
    n_rad: int
    n_cls: int
    w0: int
    S_band: np.ndarray       # [n_cls, n_rad, 2*w0+1] complex128
    H0_band: np.ndarray      # [n_cls, n_rad, 2*w0+1] complex128
    cls_of_chan: np.ndarray  # [n_ang] int32
    terms: List[Term]
    dt: float
    rtol: float
    max_iter: int
    n_steps: int
    g_of_t: Callable[[float], np.ndarray]   # t -> [n_terms] real
    c0: np.ndarray           # [n_ang*n_rad] complex128
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return self.n_ang * self.n_rad

    @property
    def n_terms(self) -> int:
        return len(self.terms)

    def g_mid(self, step: int, dt: float | None = None) -> np.ndarray:
        """Field coefficients at the midpoint t_{n+1/2} = (n + 1/2) dt (Eq. 22)."""
        dt = self.dt if dt is None else dt
        return np.asarray(self.g_of_t((step + 0.5) * dt), dtype=np.float64).reshape(self.n_terms)

    def g_table(self, n_steps: int | None = None, first_step: int = 0) -> np.ndarray:
        n_steps = self.n_steps if n_steps is None else n_steps
        out = np.empty((n_steps, self.n_terms), dtype=np.float64)
        for s in range(n_steps):
            out[s] = self.g_mid(first_step + s)
        return out


def band_to_dense(band: np.ndarray) -> np.ndarray:
    """Expand ``band[i, d+w] = R[i, i+d]`` to a dense (n, n) array (format conversion only)."""
    n, nd = band.shape
    w = (nd - 1) // 2
    out = np.zeros((n, n), dtype=band.dtype)
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(n, n - d)
        idx = np.arange(lo, hi)
        out[idx, idx + d] = band[idx, d + w]
    return out


def dense_to_band(mat: np.ndarray, w: int) -> np.ndarray:
    """Pack the 2w+1 central diagonals of a dense matrix into the row-major band layout."""
    n = mat.shape[0]
    band = np.zeros((n, 2 * w + 1), dtype=np.complex128)
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(n, n - d)
        idx = np.arange(lo, hi)
        band[idx, d + w] = mat[idx, idx + d]
    return band
