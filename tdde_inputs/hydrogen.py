"""Hydrogen-like Dirac problem in the paper's basis (BASELINE.json configs[1]).

What is built (CPU, setup only -- the paper's "pre-computation of the input data",
PAPER.md:253-256):

* B-splines of order k on evenly spaced breakpoints with repeated end knots,
  by the Cox-de Boor recursion (Eq. 10-11); the first and the
  last spline are discarded (reading R7 of PAPER.md:165);
* dual-kinetic-balance radial functions (Eq. 12-13);
* the radial Dirac operator with the paper's shifted beta,
  integrated by Gauss-Legendre quadrature per knot interval;
  H0 and S blocks per kappa;
* the dipole-limit, z-polarised interaction -c alpha_z A(t) (Eq. 4 with
  Eq. 14 at r -> 0) written as Kronecker terms A_L (x) R_L with the
  g0 + kappa' g1 + kappa g2 + kappa' kappa g3 split of PAPER.md:155-159 (Eq. 17).

Output is a ``Problem`` in the boundary layout with the two radial components
interleaved (j = 2 m + comp), which turns the three-band block of PAPER.md:126-130
(Fig. 1) into one band of half-width 2(k-1)+1.
"""
from __future__ import annotations

import math

import numpy as np

from .problem import Problem, Term, dense_to_band

C_LIGHT = 137.035999084   # DESIGN.md reading R8 (paper silent)


# ----------------------------------------------------------------------------- B-splines
def knot_vector(n_break: int, r_max: float, order: int) -> np.ndarray:
    brk = np.linspace(0.0, r_max, n_break)
    return np.concatenate([np.zeros(order - 1), brk, np.full(order - 1, r_max)])


def bspline_table(t: np.ndarray, order: int, x: np.ndarray):
    """All B-splines of the given order at points x (strictly inside knot intervals):
    returns (B, dB, d2B), each [len(x), n_splines].  Cox-de Boor, PAPER.md:109-114 (Eq. 10-11);
    derivatives from the standard difference formula of the same recursion."""
    p = order - 1
    nk = len(t)
    span = np.searchsorted(t, x, side="right") - 1          # t[span] <= x < t[span+1]
    N = [np.zeros((len(x), nk - 1))]
    N[0][np.arange(len(x)), span] = 1.0
    for d in range(1, p + 1):
        nb = nk - 1 - d
        Nd = np.zeros((len(x), nb))
        for i in range(nb):
            d1 = t[i + d] - t[i]
            d2 = t[i + d + 1] - t[i + 1]
            if d1 > 0.0:
                Nd[:, i] += (x - t[i]) / d1 * N[d - 1][:, i]
            if d2 > 0.0:
                Nd[:, i] += (t[i + d + 1] - x) / d2 * N[d - 1][:, i + 1]
        N.append(Nd)

    def deriv(lower: np.ndarray, d: int) -> np.ndarray:
        """derivative-like combination: d * (lower_i/(t_{i+d}-t_i) - lower_{i+1}/(t_{i+d+1}-t_{i+1}))"""
        nb = nk - 1 - d
        out = np.zeros((len(x), nb))
        for i in range(nb):
            d1 = t[i + d] - t[i]
            d2 = t[i + d + 1] - t[i + 1]
            if d1 > 0.0:
                out[:, i] += d * lower[:, i] / d1
            if d2 > 0.0:
                out[:, i] -= d * lower[:, i + 1] / d2
        return out

    B = N[p]
    dB = deriv(N[p - 1], p)
    d2B = deriv(deriv(N[p - 2], p - 1), p)
    return B, dB, d2B


def gauss_points(t: np.ndarray, n_gauss: int):
    xg, wg = np.polynomial.legendre.leggauss(n_gauss)
    brk = np.unique(t)
    a, b = brk[:-1], brk[1:]
    x = (0.5 * (b - a))[:, None] * xg[None, :] + (0.5 * (a + b))[:, None]
    w = (0.5 * (b - a))[:, None] * wg[None, :]
    return x.ravel(), w.ravel()


# ----------------------------------------------------------------------------- radial part
def radial_tables(n_r: int, r_max: float, order: int, n_gauss: int, c: float):
    """Quadrature tables of the kappa-independent pieces of the DKB functions (Eq. 12-13):
    P = P0 + kappa P1, Q = Q0 + kappa Q1, dP/dr = dP0 + kappa dP1, components interleaved."""
    n_break = n_r + 4 - order                  # n_splines = n_break + order - 2 = n_r + 2
    t = knot_vector(n_break, r_max, order)
    x, wq = gauss_points(t, n_gauss)
    B, dB, d2B = bspline_table(t, order, x)
    assert B.shape[1] == n_r + 2
    u, du, d2u = B[:, 1:-1], dB[:, 1:-1], d2B[:, 1:-1]    # drop first and last spline
    r = x[:, None]
    n_rad = 2 * n_r
    z = np.zeros_like(u)

    def il(c0, c1):               # interleave: column 2m <- comp 0 (Eq. 12), 2m+1 <- comp 1 (Eq. 13)
        out = np.empty((len(x), n_rad))
        out[:, 0::2], out[:, 1::2] = c0, c1
        return out

    tab = dict(
        P0=il(u, du / (2 * c)),              P1=il(z, -u / (2 * c * r)),
        Q0=il(du / (2 * c), u),              Q1=il(u / (2 * c * r), z),
        dP0=il(du, d2u / (2 * c)),           dP1=il(z, (-du / r + u / r ** 2) / (2 * c)),
    )
    return x, wq, tab


def radial_blocks(kappa: int, x, wq, tab, Z: float, c: float):
    """Dense S_kappa and H0_kappa: symmetric bilinear form of the radial Dirac operator with
    V = -Z/r, large-component rest energy 0 and small-component -2c^2."""
    P = tab["P0"] + kappa * tab["P1"]
    Q = tab["Q0"] + kappa * tab["Q1"]
    dP = tab["dP0"] + kappa * tab["dP1"]
    V = -Z / x
    W = wq[:, None]
    S = P.T @ (W * P) + Q.T @ (W * Q)
    H = P.T @ ((wq * V)[:, None] * P) + Q.T @ ((wq * (V - 2 * c * c))[:, None] * Q)
    X1 = dP.T @ (W * Q)
    H += c * (X1 + X1.T)
    X2 = P.T @ ((wq / x)[:, None] * Q)
    H += c * kappa * (X2 + X2.T)
    return 0.5 * (S + S.T), 0.5 * (H + H.T)


# ----------------------------------------------------------------------------- angular part
def l_of_kappa(kappa: int) -> int:
    return kappa if kappa > 0 else -kappa - 1


def sigma_z_element(k1: int, k2: int, mu: float) -> float:
    """<chi_{k1,mu}| sigma_z |chi_{k2,mu}> for spherical spinors (Eq. 8 with the usual
    Clebsch-Gordan phases); non-zero only when both share the orbital l."""
    if k1 == 0 or k2 == 0 or abs(mu) > abs(k1) - 0.5 + 1e-12 or abs(mu) > abs(k2) - 0.5 + 1e-12:
        return 0.0
    if k1 == k2:
        return -2.0 * mu / (2 * k1 + 1)
    if k2 == -k1 - 1:
        l = l_of_kappa(k1)
        return -2.0 * math.sqrt(max((l + 0.5) ** 2 - mu * mu, 0.0)) / (2 * l + 1)
    return 0.0


def channel_list(kappa_max: int):
    """kappa = -1,+1,-2,+2,...; each with ascending mu (reading R9)."""
    kappas = []
    for mag in range(1, kappa_max + 1):
        kappas += [-mag, mag]
    chans, cls_of_chan = [], []
    for k_idx, kap in enumerate(kappas):
        j = abs(kap) - 0.5
        mu = -j
        while mu <= j + 1e-12:
            chans.append((kap, mu))
            cls_of_chan.append(k_idx)
            mu += 1.0
    return kappas, chans, np.asarray(cls_of_chan, dtype=np.int32)


def dense_to_csr(A: np.ndarray):
    n = A.shape[0]
    rowptr = np.zeros(n + 1, dtype=np.int32)
    cols, vals = [], []
    for a in range(n):
        nz = np.nonzero(A[a])[0]
        cols += list(nz)
        vals += list(A[a, nz])
        rowptr[a + 1] = len(cols)
    return rowptr, np.asarray(cols, dtype=np.int32), np.asarray(vals, dtype=np.complex128)


# ----------------------------------------------------------------------------- pulse
def pulse_A(t: float, e0: float, omega: float, n_cycles: float) -> float:
    """A(t) of Eq. 14 at r -> 0: (E0/omega) sin^2(pi t/T) sin(omega t) on 0 < t < T."""
    T = 2.0 * math.pi * n_cycles / omega
    if t <= 0.0 or t >= T:
        return 0.0
    return e0 / omega * math.sin(math.pi * t / T) ** 2 * math.sin(omega * t)


# ----------------------------------------------------------------------------- problem
def make_hydrogen(n_r: int = 200, r_max: float = 100.0, order: int = 7, kappa_max: int = 4,
                  Z: float = 1.0, c: float = C_LIGHT, n_gauss: int = 14, e0: float = 0.05,
                  omega: float = 0.057, n_cycles: float = 3.0, dt: float = 0.01, n_steps: int = 100,
                  rtol: float = 1e-10, max_iter: int = 200, field: bool = True,
                  t_offset: float = 0.0) -> Problem:
    x, wq, tab = radial_tables(n_r, r_max, order, n_gauss, c)
    n_rad = 2 * n_r
    w = 2 * (order - 1) + 1
    kappas, chans, cls_of_chan = channel_list(kappa_max)
    n_ang, n_cls = len(chans), len(kappas)

    S_band = np.zeros((n_cls, n_rad, 2 * w + 1), dtype=np.complex128)
    H0_band = np.zeros_like(S_band)
    dense = {}
    for k_idx, kap in enumerate(kappas):
        S, H = radial_blocks(kap, x, wq, tab, Z, c)
        dense[kap] = (S, H)
        S_band[k_idx] = dense_to_band(S, w)
        H0_band[k_idx] = dense_to_band(H, w)

    # radial coupling matrices g^n[i, j] of Eq. 17: int P_i^{kappa'} Q_j^{kappa} dr = g0 + k' g1 + k g2 + k' k g3
    W = wq[:, None]
    g = [tab["P0"].T @ (W * tab["Q0"]), tab["P1"].T @ (W * tab["Q0"]),
         tab["P0"].T @ (W * tab["Q1"]), tab["P1"].T @ (W * tab["Q1"])]

    # angular factors: a1[c', c] = <k' mu| sigma_z |-k mu>, a2[c', c] = <-k' mu| sigma_z |k mu>, mu conserved
    a1 = np.zeros((n_ang, n_ang))
    a2 = np.zeros((n_ang, n_ang))
    for i, (kp, mup) in enumerate(chans):
        for j, (k, mu) in enumerate(chans):
            if abs(mup - mu) > 1e-12:
                continue
            a1[i, j] = sigma_z_element(kp, -k, mu)
            a2[i, j] = sigma_z_element(-kp, k, mu)
    K = np.diag([float(kp) for kp, _ in chans])

    # H_I = -c alpha_z A(t);  <psi'|alpha_z|psi> = i a1 int P'Q - i a2 int Q'P
    ang = [(-1j * c) * a1, (-1j * c) * (K @ a1), (-1j * c) * (a1 @ K), (-1j * c) * (K @ a1 @ K),
           (+1j * c) * a2, (+1j * c) * (K @ a2), (+1j * c) * (a2 @ K), (+1j * c) * (K @ a2 @ K)]
    rad = [g[0], g[1], g[2], g[3], g[0].T, g[2].T, g[1].T, g[3].T]
    terms = []
    for A, R in zip(ang, rad):
        rowptr, col, val = dense_to_csr(A)
        terms.append(Term(w=w, R_band=dense_to_band(R, w), A_rowptr=rowptr, A_col=col, A_val=val))

    if field:
        def g_of_t(t, _n=len(terms)):
            return np.full(_n, pulse_A(t + t_offset, e0, omega, n_cycles))
    else:
        def g_of_t(t, _n=len(terms)):
            return np.zeros(_n)

    c0 = np.zeros(n_ang * n_rad, dtype=np.complex128)   # filled by the caller (e.g. with an eigenstate)
    return Problem(name="hydrogen", n_ang=n_ang, n_rad=n_rad, n_cls=n_cls, w0=w, S_band=S_band,
                   H0_band=H0_band, cls_of_chan=cls_of_chan, terms=terms, dt=dt, rtol=rtol,
                   max_iter=max_iter, n_steps=n_steps, g_of_t=g_of_t, c0=c0, seed=0,
                   meta=dict(kappas=kappas, chans=chans, dense=dense, Z=Z, c=c, order=order,
                             n_r=n_r, r_max=r_max, a1=a1, a2=a2, g=g))
