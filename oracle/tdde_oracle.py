"""ORACLE -- test infrastructure, not product code.

A plain, slow CPU statement (NumPy / SciPy, complex FP64) of what the GPU hot path
computes: the implicit Crank-Nicolson step of the time-dependent Dirac equation,

    (S + i dt/2 H(t_{n+1/2})) c^{n+1} = (S - i dt/2 H(t_{n+1/2})) c^n       PAPER.md:209 (Eq. 25),
                                                                             midpoint: PAPER.md:195 (Eq. 22)
    H(t) = H0 + sum_L g_L(t) (A_L (x) R_L)                                   PAPER.md:155-161 (Eq. 17)

solved by BiCGSTAB preconditioned with the LU factors of
M = S + i dt/2 H0 (Eq. 26).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It shares no code with the CUDA path and does not
import it.  Operators are assembled explicitly in CSR by index loops; the solver is
the textbook preconditioned BiCGSTAB in the order and notation of DESIGN.md
"Readings" R5; the preconditioner solve is LAPACK zgbtrf/zgbtrs.

Pins (tests/test_oracle_pins.py): dense LU solve of the same system, Cayley-transform
S-norm conservation, exact CN phase of field-free eigenstates, time reversal,
closed-form hydrogen energies, Kronecker identities, LAPACK band solve; the panel-streamed
apply (apply_panels, cn_step_panels) against numpy.kron dense operators and the CSR apply.
Parity unpinned: BiCGSTAB iteration *counts* (nothing in the paper fixes them).
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Optional

import numpy as np
import scipy.sparse as sp
from scipy.linalg import lapack

TINY = 1e-290   # breakdown safeguard, reading R5


# ----------------------------------------------------------------------------- assembly (C1, C2)
def _band_coo(band: np.ndarray, row0: int, col0: int, scale: complex = 1.0):
    """COO triplets of one radial band block placed at (row0, col0): R[i, i+d] = band[i, d+w]."""
    n_rad, nd = band.shape
    w = (nd - 1) // 2
    rows, cols, vals = [], [], []
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(n_rad, n_rad - d)
        i = np.arange(lo, hi)
        rows.append(row0 + i)
        cols.append(col0 + i + d)
        vals.append(scale * band[lo:hi, d + w])
    return np.concatenate(rows), np.concatenate(cols), np.concatenate(vals)


def _to_csr(rows, cols, vals, n):
    m = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(n, n))
    m = m.tocsr()            # sums duplicates
    m.sort_indices()
    return m


def assemble_block_diagonal(band_per_cls: np.ndarray, cls_of_chan: np.ndarray, n_ang: int, n_rad: int):
    """S or H0: block (a, a) is the band of class cls_of_chan[a] (PAPER.md:161 delta_{k'k} delta_{m'm}; :180)."""
    rows, cols, vals = [], [], []
    for a in range(n_ang):
        r, c, v = _band_coo(band_per_cls[cls_of_chan[a]], a * n_rad, a * n_rad)
        rows.append(r), cols.append(c), vals.append(v)
    return _to_csr(rows, cols, vals, n_ang * n_rad)


def assemble_kron_term(term, n_ang: int, n_rad: int):
    """K_L[I(a',i), I(a,j)] = A_L[a', a] R_L[i, j]: loop over the non-zeros of A_L, place one band block each."""
    rows, cols, vals = [], [], []
    for ap in range(n_ang):
        for k in range(term.A_rowptr[ap], term.A_rowptr[ap + 1]):
            a = int(term.A_col[k])
            r, c, v = _band_coo(term.R_band, ap * n_rad, a * n_rad, scale=term.A_val[k])
            rows.append(r), cols.append(c), vals.append(v)
    if not rows:
        return sp.csr_matrix((n_ang * n_rad, n_ang * n_rad), dtype=np.complex128)
    return _to_csr(rows, cols, vals, n_ang * n_rad)


@dataclass
class Operators:
    n_ang: int
    n_rad: int
    S: sp.csr_matrix
    H0: sp.csr_matrix
    K: List[sp.csr_matrix]

    @property
    def n(self):
        return self.n_ang * self.n_rad


def assemble(problem) -> Operators:
    S = assemble_block_diagonal(problem.S_band, problem.cls_of_chan, problem.n_ang, problem.n_rad)
    H0 = assemble_block_diagonal(problem.H0_band, problem.cls_of_chan, problem.n_ang, problem.n_rad)
    K = [assemble_kron_term(t, problem.n_ang, problem.n_rad) for t in problem.terms]
    return Operators(problem.n_ang, problem.n_rad, S, H0, K)


def hamiltonian_csr(ops: Operators, g: np.ndarray) -> sp.csr_matrix:
    """H(t) = H0 + sum_L g_L K_L as one CSR matrix (the paper re-values H each step)."""
    H = ops.H0.copy()
    for gl, KL in zip(g, ops.K):
        if gl != 0.0:
            H = H + gl * KL
    return H.tocsr()


def apply_H(ops: Operators, g: np.ndarray, x: np.ndarray) -> np.ndarray:
    y = ops.H0 @ x
    for gl, KL in zip(g, ops.K):
        if gl != 0.0:
            y = y + gl * (KL @ x)
    return y


def apply(ops: Operators, alpha: complex, beta: complex, g: np.ndarray, x: np.ndarray) -> np.ndarray:
    """y = alpha S x + beta (H0 + sum_L g_L A_L (x) R_L) x   (the tdde_apply export)."""
    return alpha * (ops.S @ x) + beta * apply_H(ops, g, x)


def s_norm_sq(ops: Operators, c: np.ndarray) -> float:
    """Re(c^H S c): total probability in the non-orthogonal basis (S: PAPER.md:178-182); reading R14."""
    return float(np.real(np.vdot(c, ops.S @ c)))


def eigenstates(problem):
    """Field-free eigenstates per kappa-class: H0_k psi = E S_k psi (Eq. 19-20 with reading R3), by LAPACK's
    generalised Hermitian-definite solver on the dense blocks.  Returns E [n_cls, n_rad] ascending and V [n_cls, n_rad, n_rad] with
    V[k, e, :] the S-orthonormal eigenvector of E[k, e]."""
    import scipy.linalg as sla
    dense = lambda band: sum(np.diag(band[max(0, -d):band.shape[0] - max(0, d), d + (band.shape[1] - 1) // 2], d)
                             for d in range(-(band.shape[1] - 1) // 2, (band.shape[1] - 1) // 2 + 1))
    E = np.zeros((problem.n_cls, problem.n_rad))
    V = np.zeros((problem.n_cls, problem.n_rad, problem.n_rad), dtype=np.complex128)
    for k in range(problem.n_cls):
        E[k], vec = sla.eigh(dense(problem.H0_band[k]), dense(problem.S_band[k]))
        V[k] = vec.T
    return E, V


def project(problem, V: np.ndarray, c: np.ndarray) -> np.ndarray:
    """P[a, e] = |<psi_{k(a), e} | Psi_a>|^2 = |v_e^H S_k c_a|^2, the terms of dP/dE (Eq. 33) before the sum over
    (kappa, mu); V[k, e, :] are eigenvectors of the field-free pencil (H0_k, S_k) (Eq. 19-20)."""
    from_band = lambda band: sum(np.diag(band[max(0, -d):band.shape[0] - max(0, d), d + (band.shape[1] - 1) // 2], d)
                                 for d in range(-(band.shape[1] - 1) // 2, (band.shape[1] - 1) // 2 + 1))
    C = c.reshape(problem.n_ang, problem.n_rad)
    out = np.zeros((problem.n_ang, V.shape[1]))
    for k in range(problem.n_cls):
        Sk = from_band(problem.S_band[k])
        idx = np.nonzero(problem.cls_of_chan == k)[0]
        amp = (V[k].conj() @ (Sk @ C[idx].T))            # [n_states, channels of the class]
        out[idx] = (np.abs(amp) ** 2).T
    return out


# ----------------------------------------------------------------------------- sampled rows (P10)
def apply_rows_sampled(problem, alpha: complex, beta: complex, g: np.ndarray, x: np.ndarray,
                       chan: np.ndarray, rad: np.ndarray) -> np.ndarray:
    """Entries (chan[s], rad[s]) of y = alpha S x + beta (H0 + sum g_L A_L (x) R_L) x by direct
    summation of the definition (C2) -- for sizes where the CSR cannot be held."""
    n_rad = problem.n_rad
    X = x.reshape(problem.n_ang, n_rad)
    out = np.zeros(len(chan), dtype=np.complex128)
    w0 = problem.w0
    for s in range(len(chan)):
        ap, i = int(chan[s]), int(rad[s])
        k = problem.cls_of_chan[ap]
        acc = 0.0 + 0.0j
        for d in range(-w0, w0 + 1):
            j = i + d
            if 0 <= j < n_rad:
                acc += (alpha * problem.S_band[k, i, d + w0] + beta * problem.H0_band[k, i, d + w0]) * X[ap, j]
        for L, term in enumerate(problem.terms):
            if g[L] == 0.0:
                continue
            w = term.w
            lo, hi = max(0, i - w), min(n_rad, i + w + 1)
            rrow = term.R_band[i, lo - i + w:hi - i + w]
            tsum = 0.0 + 0.0j
            for kk in range(term.A_rowptr[ap], term.A_rowptr[ap + 1]):
                a = int(term.A_col[kk])
                tsum += term.A_val[kk] * np.dot(rrow, X[a, lo:hi])
            acc += beta * g[L] * tsum
        out[s] = acc
    return out


# ----------------------------------------------------------------------------- panel-streamed apply (P10, full vector)
def _band_times_rows(band: np.ndarray, X: np.ndarray) -> np.ndarray:
    """U[c, i] = sum_d band[i, d+w] X[c, i+d]  (one radial band matrix applied to every row-vector X[c, :])."""
    n_rad, nd = band.shape
    w = (nd - 1) // 2
    U = np.zeros_like(X)
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(n_rad, n_rad - d)
        U[:, lo:hi] += band[lo:hi, d + w][None, :] * X[:, lo + d:hi + d]
    return U


def apply_panels(problem, alpha: complex, beta: complex, g: np.ndarray, x: np.ndarray, panel: int = 256) -> np.ndarray:
    """y = alpha S x + beta (H0 + sum_L g_L A_L (x) R_L) x for sizes where the CSR cannot be held, evaluated
    from the definition (Eq. 17) one panel of `panel` output channels at a
    time: for output channel a' the block part is the class band of a' applied to x[a', :], and each coupling
    term is sum_a A_L[a', a] (R_L x[a, :]) -- the radial band first, then the angular sum over the non-zeros of
    row a' of A_L.  No assembled matrix, no operand larger than (panel + coupled channels) x n_rad."""
    n_ang, n_rad = problem.n_ang, problem.n_rad
    X = np.ascontiguousarray(x).reshape(n_ang, n_rad)
    Y = np.zeros_like(X)
    for a0 in range(0, n_ang, panel):
        a1 = min(n_ang, a0 + panel)
        for k in np.unique(problem.cls_of_chan[a0:a1]):
            idx = a0 + np.nonzero(problem.cls_of_chan[a0:a1] == k)[0]
            Y[idx] += _band_times_rows(alpha * problem.S_band[k] + beta * problem.H0_band[k], X[idx])
        for L, term in enumerate(problem.terms):
            if g[L] == 0.0:
                continue
            lo, hi = int(term.A_rowptr[a0]), int(term.A_rowptr[a1])
            if hi == lo:
                continue
            cols = np.unique(term.A_col[lo:hi])                      # channels coupled to this panel by A_L
            U = _band_times_rows(term.R_band, X[cols])               # R_L x[a, :] for those channels
            where = {int(c): q for q, c in enumerate(cols)}
            for ap in range(a0, a1):
                for kk in range(term.A_rowptr[ap], term.A_rowptr[ap + 1]):
                    Y[ap] += (beta * g[L] * term.A_val[kk]) * U[where[int(term.A_col[kk])]]
    return Y.reshape(-1)


# ----------------------------------------------------------------------------- preconditioner (C5)
@dataclass
class PrecondFactors:
    n_ang: int
    n_rad: int
    w0: int
    cls_of_chan: np.ndarray
    lu: list       # per class: LAPACK zgbtrf band factor
    piv: list


def factor_precond(problem, dt: Optional[float] = None) -> PrecondFactors:
    """LU of M_k = S_k + i dt/2 H0_k per kappa-class (Eq. 26), LAPACK zgbtrf with pivoting."""
    dt = problem.dt if dt is None else dt
    tau = 0.5 * dt
    w, n_rad = problem.w0, problem.n_rad
    lus, pivs = [], []
    for k in range(problem.n_cls):
        Mb = problem.S_band[k] + 1j * tau * problem.H0_band[k]      # [n_rad, 2w+1], Mb[i, d+w] = M[i, i+d]
        ab = np.zeros((3 * w + 1, n_rad), dtype=np.complex128)      # LAPACK: ab[kl+ku+i-j, j] = M[i, j]
        for d in range(-w, w + 1):
            lo, hi = max(0, -d), min(n_rad, n_rad - d)
            i = np.arange(lo, hi)
            ab[2 * w - d, i + d] = Mb[i, d + w]
        lu, piv, info = lapack.zgbtrf(ab, w, w)
        if info != 0:
            raise np.linalg.LinAlgError(f"zgbtrf info={info} for class {k}")
        lus.append(lu), pivs.append(piv)
    return PrecondFactors(problem.n_ang, n_rad, w, problem.cls_of_chan.copy(), lus, pivs)


def apply_precond(f: PrecondFactors, x: np.ndarray) -> np.ndarray:
    """y = M^{-1} x, block-Jacobi over angular channels (M is block-diagonal: PAPER.md:211-215)."""
    X = x.reshape(f.n_ang, f.n_rad)
    Y = np.empty_like(X)
    for k in range(len(f.lu)):
        idx = np.nonzero(f.cls_of_chan == k)[0]
        if len(idx) == 0:
            continue
        rhs = np.asfortranarray(X[idx].T)
        sol, info = lapack.zgbtrs(f.lu[k], f.w0, f.w0, rhs, f.piv[k])
        if info != 0:
            raise np.linalg.LinAlgError(f"zgbtrs info={info}")
        Y[idx] = sol.T
    return Y.reshape(-1)


# ----------------------------------------------------------------------------- BiCGSTAB (C4)
@dataclass
class SolveInfo:
    half_iters: int          # a full iteration counts 2; the half-step exit leaves an odd count
    converged: bool
    status: str              # "ok" | "breakdown" | "noconv"
    rel_res: float
    applies: int
    trace: Optional[list] = None


def _bad(z) -> bool:
    return (not np.isfinite(z)) or abs(z) < TINY


def bicgstab(A_mul, M_solve, b: np.ndarray, x0: np.ndarray, rtol: float, max_iter: int,
             force_iters: Optional[int] = None, keep_trace: bool = False):
    """Preconditioned BiCGSTAB, step for step as in DESIGN.md R5 / SURVEY.md C4 (van der Vorst's
    form with K = M applied on the right; r is the residual of the original system).

    force_iters=k disables every exit test and runs exactly k full iterations (pin P11)."""
    vdot = np.vdot                                   # <u, v> = sum conj(u_i) v_i
    x = x0.copy()
    r = b - A_mul(x)
    rhat = r.copy()
    nb = np.linalg.norm(b)
    applies = 1
    trace = [] if keep_trace else None
    res = np.linalg.norm(r)
    if force_iters is None and res <= rtol * nb:
        return x, SolveInfo(0, True, "ok", res / nb if nb > 0 else 0.0, applies, trace)
    rho_old = alpha = omega = 1.0 + 0.0j
    v = np.zeros_like(x)
    p = np.zeros_like(x)
    n_iter = max_iter if force_iters is None else force_iters
    half = 0
    for _k in range(1, n_iter + 1):
        rho = vdot(rhat, r)
        if _bad(rho):
            return x, SolveInfo(half, False, "breakdown", res / nb, applies, trace)
        beta = (rho / rho_old) * (alpha / omega)
        rho_old = rho
        p = r + beta * (p - omega * v)
        y = M_solve(p)
        v = A_mul(y)
        applies += 1
        rv = vdot(rhat, v)
        if _bad(rv):
            return x, SolveInfo(half, False, "breakdown", res / nb, applies, trace)
        alpha = rho / rv
        s = r - alpha * v
        half += 1
        res = np.linalg.norm(s)
        if force_iters is None and res <= rtol * nb:
            x = x + alpha * y
            return x, SolveInfo(half, True, "ok", res / nb, applies, trace)
        z = M_solve(s)
        t = A_mul(z)
        applies += 1
        tt = vdot(t, t)
        if _bad(tt):
            return x, SolveInfo(half, False, "breakdown", res / nb, applies, trace)
        omega = vdot(t, s) / tt
        x = x + alpha * y + omega * z
        r = s - omega * t
        half += 1
        res = np.linalg.norm(r)
        if keep_trace:
            trace.append(dict(p=p.copy(), v=v.copy(), s=s.copy(), t=t.copy(), x=x.copy(), r=r.copy(),
                              y=y.copy(), z=z.copy(), alpha=alpha, omega=omega, rho=rho, beta=beta))
        if force_iters is None and res <= rtol * nb:
            return x, SolveInfo(half, True, "ok", res / nb, applies, trace)
    if force_iters is not None:
        return x, SolveInfo(half, True, "ok", res / nb, applies, trace)
    return x, SolveInfo(half, False, "noconv", res / nb, applies, trace)


# ----------------------------------------------------------------------------- Crank-Nicolson (C3)
def cn_step(ops: Operators, fact: PrecondFactors, c: np.ndarray, g_mid: np.ndarray, dt: float,
            rtol: float, max_iter: int, assembled: bool = True, force_iters: Optional[int] = None,
            keep_trace: bool = False):
    """One step of Eq. 25 with H at the midpoint (Eq. 22): A = S + i tau H, B = S - i tau H, solve A x = B c,
    x0 = c (reading R5)."""
    tau = 0.5 * dt
    if assembled:
        H = hamiltonian_csr(ops, g_mid)
        A = (ops.S + 1j * tau * H).tocsr()
        B = (ops.S - 1j * tau * H).tocsr()
        A_mul = lambda u: A @ u
        b = B @ c
    else:
        A_mul = lambda u: ops.S @ u + 1j * tau * apply_H(ops, g_mid, u)
        b = ops.S @ c - 1j * tau * apply_H(ops, g_mid, c)
    M_solve = lambda u: apply_precond(fact, u)
    return bicgstab(A_mul, M_solve, b, c, rtol, max_iter, force_iters=force_iters, keep_trace=keep_trace)


def cn_step_panels(problem, fact: PrecondFactors, c: np.ndarray, g_mid: np.ndarray, dt: float, rtol: float,
                   max_iter: int, panel: int = 256):
    """cn_step for sizes where the CSR cannot be held: the same A, B and the same bicgstab, with every product
    evaluated by apply_panels (A = S + i tau H: alpha = 1, beta = +i tau; B: beta = -i tau)."""
    tau = 0.5 * dt
    A_mul = lambda u: apply_panels(problem, 1.0, 1j * tau, g_mid, u, panel)
    b = apply_panels(problem, 1.0, -1j * tau, g_mid, c, panel)
    M_solve = lambda u: apply_precond(fact, u)
    return bicgstab(A_mul, M_solve, b, c, rtol, max_iter)


def propagate(problem, ops: Operators, fact: PrecondFactors, c0: np.ndarray, n_steps: int,
              first_step: int = 0, dt: Optional[float] = None, assembled: bool = True):
    """c^{n+1} from c^n for n_steps steps; g_L sampled at t_{n+1/2} = (n + 1/2) dt."""
    dt = problem.dt if dt is None else dt
    c = c0.copy()
    infos = []
    for s in range(n_steps):
        g = problem.g_mid(first_step + s, dt)
        c, info = cn_step(ops, fact, c, g, dt, problem.rtol, problem.max_iter, assembled=assembled)
        infos.append(info)
        if info.status != "ok":
            break
    return c, infos
