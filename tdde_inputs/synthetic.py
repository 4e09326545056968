"""Seeded synthetic workloads shaped like the paper's (BASELINE.json configs).

The paper measures on its own hydrogen/laser matrices, which
are not available; these inputs take their *structure*: block-diagonal H0 / S
with kappa-dependent banded radial blocks, coupling = sum of
(sparse angular) (x) (banded radial) terms with scalar time factors
(Eq. 17), complex FP64.

All random numbers come from ``numpy.random.default_rng(seed)`` and are drawn in
this order: H0 base band, H0 second band, then for L = 0..T-1: R_L then A_L, then
the initial vector c0.
"""
from __future__ import annotations

import math

import numpy as np

from .problem import Problem, Term

E0_DEFAULT = 0.05
OMEGA_DEFAULT = 0.057

# name -> generator arguments; BASELINE.json "configs" in order (hydrogen is in hydrogen.py)
CONFIGS = {
    "tiny":   dict(n_ang=16,   n_r=64,   bandwidth=7,  n_terms=3, tiny_offsets=True,
                   dt=0.01,  n_steps=10,  rtol=1e-12, seed=0),
    "medium": dict(n_ang=512,  n_r=500,  bandwidth=13, n_terms=5, dt=0.005, n_steps=100, rtol=1e-10, seed=1),
    "large":  dict(n_ang=3000, n_r=1000, bandwidth=13, n_terms=5, dt=0.005, n_steps=50,  rtol=1e-10, seed=2),
    "hbm":    dict(n_ang=8000, n_r=2000, bandwidth=13, n_terms=7, dt=0.002, n_steps=20,  rtol=1e-10, seed=3),
    # bandwidth sweep at HBM-scale size (BASELINE.json configs[4])
    "hbm_bw7":  dict(n_ang=8000, n_r=2000, bandwidth=7,  n_terms=7, dt=0.002, n_steps=20, rtol=1e-10, seed=3),
    "hbm_bw19": dict(n_ang=8000, n_r=2000, bandwidth=19, n_terms=7, dt=0.002, n_steps=20, rtol=1e-10, seed=3),
}


def herm_band(rng: np.random.Generator, n: int, w: int) -> np.ndarray:
    """Random Hermitian band: real N(0,1) diagonal, (N+iN)/sqrt2 super-diagonals, conjugate below."""
    band = np.zeros((n, 2 * w + 1), dtype=np.complex128)
    band[:, w] = rng.standard_normal(n)
    for d in range(1, w + 1):
        v = (rng.standard_normal(n - d) + 1j * rng.standard_normal(n - d)) / math.sqrt(2.0)
        band[: n - d, w + d] = v          # R[i, i+d]
        band[d:, w - d] = np.conj(v)      # R[i+d, i] = conj(R[i, i+d])
    return band


def spd_band(n: int, w: int, q: float = 0.3) -> np.ndarray:
    """S[i, j] = q^|i-j| inside the band (real, SPD for q = 0.3)."""
    band = np.zeros((n, 2 * w + 1), dtype=np.complex128)
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(n, n - d)
        band[lo:hi, d + w] = q ** abs(d)
    return band


def kappa_classes(n_ang: int):
    """kappa = -1,+1,-2,+2,... each owning 2|kappa| consecutive channels until n_ang."""
    kappas, cls_of_chan = [], np.empty(n_ang, dtype=np.int32)
    a, k = 0, 0
    while a < n_ang:
        mag = k // 2 + 1
        kappa = -mag if k % 2 == 0 else mag
        cnt = min(2 * mag, n_ang - a)
        cls_of_chan[a:a + cnt] = k
        kappas.append(kappa)
        a += cnt
        k += 1
    return np.asarray(kappas, dtype=np.int64), cls_of_chan


def banded_hermitian_csr(rng: np.random.Generator, n_ang: int, max_off: int):
    """Hermitian, non-periodic A with non-zeros at offsets +-1..+-max_off, CSR with sorted columns."""
    upper = {}
    for off in range(1, max_off + 1):
        m = max(n_ang - off, 0)
        upper[off] = (rng.standard_normal(m) + 1j * rng.standard_normal(m)) / math.sqrt(2.0)
    rowptr = np.zeros(n_ang + 1, dtype=np.int32)
    cols, vals = [], []
    for a in range(n_ang):
        for off in range(-max_off, max_off + 1):
            b = a + off
            if off == 0 or b < 0 or b >= n_ang:
                continue
            cols.append(b)
            vals.append(upper[off][a] if off > 0 else np.conj(upper[-off][b]))
        rowptr[a + 1] = len(cols)
    return rowptr, np.asarray(cols, dtype=np.int32), np.asarray(vals, dtype=np.complex128)


def s_norm_sq_banded(S_band: np.ndarray, cls_of_chan: np.ndarray, c: np.ndarray, n_ang: int, n_rad: int) -> float:
    """Re(c^H S c) by direct summation over band diagonals; used only to scale c0."""
    w = (S_band.shape[2] - 1) // 2
    C = c.reshape(n_ang, n_rad)
    Sb = S_band[cls_of_chan]            # [n_ang, n_rad, nd] (view per channel class)
    tot = 0.0
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(n_rad, n_rad - d)
        tot += float(np.real(np.sum(np.conj(C[:, lo:hi]) * Sb[:, lo:hi, d + w] * C[:, lo + d:hi + d])))
    return tot


def make_synthetic(n_ang: int, n_r: int, bandwidth: int, n_terms: int, dt: float, n_steps: int,
                   rtol: float, seed: int, tiny_offsets: bool = False, e0: float = E0_DEFAULT,
                   omega: float = OMEGA_DEFAULT, phase: float = 0.0, max_iter: int = 200,
                   name: str = "synthetic", with_c0: bool = True, s_q: float = 0.3, h0_scale: float = 1.0) -> Problem:
    """s_q: decay of the SPD band S[i,j] = s_q^|i-j| (0.3 in every BASELINE config; larger = worse conditioned);
    h0_scale multiplies H0 (stiff field-free blocks, tau |H0| >> |S|, as the Dirac rest-mass terms are)."""
    assert bandwidth % 2 == 1
    w = (bandwidth - 1) // 2
    n_rad = 2 * n_r
    rng = np.random.default_rng(seed)

    kappas, cls_of_chan = kappa_classes(n_ang)
    n_cls = len(kappas)
    kmax = float(np.max(np.abs(kappas)))

    S1 = spd_band(n_rad, w, s_q)
    base = herm_band(rng, n_rad, w)
    second = herm_band(rng, n_rad, w)
    S_band = np.broadcast_to(S1, (n_cls, n_rad, 2 * w + 1)).copy()
    H0_band = h0_scale * (base[None] + (kappas[:, None, None] / kmax) * second[None])

    terms = []
    for L in range(n_terms):
        R = herm_band(rng, n_rad, w)
        max_off = 2 if tiny_offsets else L + 1
        rowptr, col, val = banded_hermitian_csr(rng, n_ang, max_off)
        terms.append(Term(w=w, R_band=R, A_rowptr=rowptr, A_col=col, A_val=val))

    def g_of_t(t, _T=n_terms, _e0=e0, _om=omega, _ph=phase):
        return np.full(_T, _e0 * math.sin(_om * t + _ph), dtype=np.float64)

    if with_c0:
        n = n_ang * n_rad
        c0 = rng.standard_normal(2 * n).view(np.complex128).copy()
        nrm, blk = 0.0, 128     # blocked over channels to bound temporary memory
        for a0 in range(0, n_ang, blk):
            a1 = min(n_ang, a0 + blk)
            nrm += s_norm_sq_banded(S_band, cls_of_chan[a0:a1], c0[a0 * n_rad:a1 * n_rad], a1 - a0, n_rad)
        c0 /= math.sqrt(nrm)
    else:
        c0 = np.zeros(0, dtype=np.complex128)

    return Problem(name=name, n_ang=n_ang, n_rad=n_rad, n_cls=n_cls, w0=w, S_band=S_band,
                   H0_band=np.ascontiguousarray(H0_band), cls_of_chan=cls_of_chan, terms=terms,
                   dt=dt, rtol=rtol, max_iter=max_iter, n_steps=n_steps, g_of_t=g_of_t, c0=c0,
                   seed=seed, meta=dict(kappas=kappas, e0=e0, omega=omega, phase=phase,
                                        bandwidth=bandwidth, n_r=n_r))


def make_config(name: str, **overrides) -> Problem:
    """Build one of the BASELINE.json synthetic configs by name (see CONFIGS)."""
    args = dict(CONFIGS[name])
    args.update(overrides)
    return make_synthetic(name=name, **args)
