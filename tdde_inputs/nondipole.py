"""Paper-shaped operator set beyond the dipole limit (SURVEY.md 8(f) NEXT-1; PAPER.md:142-147 Eq. 15, :155-170 Eq. 17-18,
:217-245 Eq. 27-30): an x-polarised pulse travelling along z couples (kappa, mu) to (kappa', mu +- 1) through

    (H^theta_l)_{k' k m' m} = 4 pi Y_l0(z^) < X_{-k', m'} | sigma_x Y_l0(r^) | X_{k, m} >                      (Eq. 18)

and the time-dependent Hamiltonian is

    H(t) = H0 + i sum_alpha f_alpha(t) sum_l { H^theta_l[k',k,m',m] [g0 + k' g1 + k g2 + k' k g3]_{alpha,l}
                                              - H^theta_l[k,k',m,m'] [g0^+ + k g1^+ + k' g2^+ + k' k g3^+]_{alpha,l} }     (Eq. 17)

What is built here, and from what:

* the ANGULAR matrices H^theta_l exactly as the paper defines them: spherical spinors from Clebsch-Gordan coefficients
  (Racah's formula, written out below), sigma_x flips the spin projection, the three-Y integral is Eq. 28's product of two
  Wigner 3j symbols.  Eq. 27 as printed has spherical-harmonic orders that do not match its Clebsch-Gordan factors; Eq. 18 is
  taken as the definition and expanded directly (reading R17).  The selection rules mu = mu' +- 1 and the
  l-triangle rule of Eq. 29-30 come out as the zero pattern (pinned in tests/test_oracle_pins.py);
* every Kronecker term of Eq. 17: (K^a H^theta_l K^b) (x) g^n_l and the adjoint bracket, K = diag(kappa): 8 terms per l;
* the field-free radial blocks H0_kappa, S_kappa of the hydrogen DKB basis (tdde_inputs.hydrogen);
* STAND-INS for what the paper only defines in its ref. [3], which is not available: the Bessel-projected radial
  matrices g^n_{alpha,l} are seeded real band matrices, taken separable in alpha (g^n_{alpha,l} = c_{alpha,l} g^n_l) so that
  the six time functions f_alpha(t) of Eq. 15 pre-combine into ONE scalar factor F_l(t) = (E0/omega) sum_alpha c_{alpha,l}
  f_alpha(t) per l (the paper pre-combines G^n_l(t) = sum_alpha f_alpha(t) g^n_{alpha,l} per step).

Nothing here applies operators or solves anything.
"""
from __future__ import annotations

import math

import numpy as np

from .hydrogen import C_LIGHT, channel_list, dense_to_csr, l_of_kappa, radial_blocks, radial_tables
from .problem import Problem, Term, dense_to_band


# ----------------------------------------------------------------------------- angular momentum algebra (doubled integers)
def _f(two_x: int) -> int:
    """(two_x / 2)! for an even, non-negative doubled argument."""
    assert two_x % 2 == 0 and two_x >= 0
    return math.factorial(two_x // 2)


def clebsch_gordan(tj1: int, tm1: int, tj2: int, tm2: int, tJ: int, tM: int) -> float:
    """<j1 m1 j2 m2 | J M> by Racah's formula; every argument is TWICE the quantum number (so half-integers are ints)."""
    if tm1 + tm2 != tM or abs(tm1) > tj1 or abs(tm2) > tj2 or abs(tM) > tJ:
        return 0.0
    if tJ < abs(tj1 - tj2) or tJ > tj1 + tj2 or (tj1 + tj2 + tJ) % 2 or (tj1 + tm1) % 2 or (tj2 + tm2) % 2 or (tJ + tM) % 2:
        return 0.0
    pref = (tJ + 1) * _f(tJ + tj1 - tj2) * _f(tJ - tj1 + tj2) * _f(tj1 + tj2 - tJ) / _f(tj1 + tj2 + tJ + 2)
    pref *= _f(tJ + tM) * _f(tJ - tM) * _f(tj1 - tm1) * _f(tj1 + tm1) * _f(tj2 - tm2) * _f(tj2 + tm2)
    tot = 0.0
    for k in range(0, (tj1 + tj2 - tJ) // 2 + 1):
        args = [tj1 + tj2 - tJ - 2 * k, tj1 - tm1 - 2 * k, tj2 + tm2 - 2 * k, tJ - tj2 + tm1 + 2 * k, tJ - tj1 - tm2 + 2 * k]
        if min(args) < 0:
            continue
        den = math.factorial(k)
        for x in args:
            den *= _f(x)
        tot += (-1) ** k / den
    return math.sqrt(pref) * tot


def wigner_3j(l1: int, l2: int, l3: int, m1: int, m2: int, m3: int) -> float:
    """(l1 l2 l3; m1 m2 m3) for integer arguments, from the Clebsch-Gordan coefficient."""
    if m1 + m2 + m3 != 0:
        return 0.0
    return (-1) ** (l1 - l2 - m3) / math.sqrt(2 * l3 + 1) * clebsch_gordan(2 * l1, 2 * m1, 2 * l2, 2 * m2, 2 * l3, -2 * m3)


def y_l0_sandwich(l1: int, m1: int, l: int, l2: int, m2: int) -> float:
    """int conj(Y_{l1 m1}) Y_{l 0} Y_{l2 m2} dOmega by Eq. 28, with conj(Y_{l m}) = (-1)^m Y_{l,-m}."""
    if m1 != m2 or abs(m1) > l1 or abs(m2) > l2:
        return 0.0
    return ((-1) ** m1 * math.sqrt((2 * l1 + 1) * (2 * l + 1) * (2 * l2 + 1) / (4.0 * math.pi))
            * wigner_3j(l1, l, l2, 0, 0, 0) * wigner_3j(l1, l, l2, -m1, 0, m2))


def spinor_cg(kappa: int, tmu: int, tms: int) -> float:
    """C(l_kappa, mu - ms; 1/2, ms | j, mu): weight of Y_{l_kappa, mu - ms} chi_{ms} in the spherical spinor X_{kappa, mu}
    (Eq. 7-8).  tmu, tms are doubled."""
    l = l_of_kappa(kappa)
    tj = 2 * abs(kappa) - 1
    return clebsch_gordan(2 * l, tmu - tms, 1, tms, tj, tmu)


def h_theta_element(l: int, kp: int, k: int, tmup: int, tmu: int) -> float:
    """(H^theta_l)_{k' k mu' mu} of Eq. 18.  sigma_x chi_{ms} = chi_{-ms}, so the bra component with spin -ms meets the ket
    component with spin ms; Y_l0(z^) = sqrt((2l+1)/4pi)."""
    lb, lk = l_of_kappa(-kp), l_of_kappa(k)
    tot = 0.0
    for tms in (-1, 1):
        tmb = tmup + tms              # 2 x (order of the bra's spherical harmonic) = 2 mu' - 2 (-ms)
        tmk = tmu - tms
        if tmb % 2 or tmk % 2:
            continue
        cb = spinor_cg(-kp, tmup, -tms)
        ck = spinor_cg(k, tmu, tms)
        if cb == 0.0 or ck == 0.0:
            continue
        tot += cb * ck * y_l0_sandwich(lb, tmb // 2, l, lk, tmk // 2)
    return 4.0 * math.pi * math.sqrt((2 * l + 1) / (4.0 * math.pi)) * tot


def h_theta(l: int, chans) -> np.ndarray:
    """Dense real H^theta_l over the channel list [(kappa, mu), ...] (rows = primed indices)."""
    n = len(chans)
    out = np.zeros((n, n))
    for i, (kp, mup) in enumerate(chans):
        for j, (k, mu) in enumerate(chans):
            tmup, tmu = int(round(2 * mup)), int(round(2 * mu))
            if abs(tmu - tmup) != 2:              # Eq. 29; everything else vanishes identically (checked by the pins)
                continue
            out[i, j] = h_theta_element(l, kp, k, tmup, tmu)
    return out


def triangle_allows(l: int, kp: int, k: int) -> bool:
    """The l-triangle and parity rule the three-Y integral imposes on (l_{-kappa'}, l, l_kappa) (Eq. 30, which the paper prints
    for the index order of the second bracket of Eq. 17)."""
    lb, lk = l_of_kappa(-kp), l_of_kappa(k)
    return abs(lb - lk) <= l <= lb + lk and (lb + l + lk) % 2 == 0


# ----------------------------------------------------------------------------- time functions
def f_alpha(t: float, omega: float, t_pulse: float) -> np.ndarray:
    """The six sine / cosine functions a sin^2 envelope times a sinusoidal carrier separates into."""
    big = 2.0 * math.pi / t_pulse
    return np.array([math.sin(omega * t), math.cos(omega * t), math.sin((omega + big) * t), math.cos((omega + big) * t),
                     math.sin((omega - big) * t), math.cos((omega - big) * t)])


# ----------------------------------------------------------------------------- problem
def make_nondipole(kappa_max: int = 6, l_max: int = 2, n_r: int = 30, r_max: float = 30.0, order: int = 7, Z: float = 1.0,
                   c: float = C_LIGHT, n_gauss: int = 14, e0: float = 0.05, omega: float = 0.5, n_cycles: float = 2.0,
                   dt: float = 0.01, n_steps: int = 20, rtol: float = 1e-10, max_iter: int = 200, seed: int = 7,
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

    rng = np.random.default_rng(seed)
    K = np.diag([float(kp) for kp, _ in chans])
    terms, l_of_term = [], []
    for l in range(l_max + 1):
        Ht = h_theta(l, chans)
        # stand-in radial matrices g^n_l: real bands of magnitude 2^-l / 2 (the projections fall off with l, PAPER.md:245;
        # c alpha . A between a large and a small DKB component is O(1) x A, as in the dipole term of tdde_inputs.hydrogen)
        gs = []
        for n in range(4):
            g = np.zeros((n_rad, n_rad))
            for d in range(-w, w + 1):
                lo, hi = max(0, -d), min(n_rad, n_rad - d)
                idx = np.arange(lo, hi)
                g[idx, idx + d] = rng.standard_normal(hi - lo)
            gs.append(g * (0.5 * 2.0 ** (-l) / (1.0 + kappa_max) ** {0: 0, 1: 1, 2: 1, 3: 2}[n]))      # kappa factors are up to kappa_max
        first = [Ht, K @ Ht, Ht @ K, K @ Ht @ K]                    # multiply g0, g1 (kappa'), g2 (kappa), g3 (kappa' kappa)
        second = [Ht.T, Ht.T @ K, K @ Ht.T, K @ Ht.T @ K]           # multiply g0^+, g1^+ (kappa = column), g2^+ (kappa' = row), g3^+
        for n in range(4):
            for A, R in ((1j * first[n], gs[n]), (-1j * second[n], gs[n].T)):
                rowptr, col, val = dense_to_csr(A)
                terms.append(Term(w=w, R_band=dense_to_band(R.astype(np.complex128), w), A_rowptr=rowptr, A_col=col, A_val=val))
                l_of_term.append(l)
    l_of_term = np.asarray(l_of_term)
    c_alpha = rng.standard_normal((6, l_max + 1)) / math.sqrt(6.0)
    t_pulse = 2.0 * math.pi * n_cycles / omega

    def g_of_t(t, _l=l_of_term):
        tt = t + t_offset
        if tt <= 0.0 or tt >= t_pulse:
            return np.zeros(len(_l))
        F = (e0 / omega) * (f_alpha(tt, omega, t_pulse) @ c_alpha)        # one factor per l
        return F[_l]

    c0 = np.zeros(n_ang * n_rad, dtype=np.complex128)
    return Problem(name="nondipole", n_ang=n_ang, n_rad=n_rad, n_cls=n_cls, w0=w, S_band=S_band, H0_band=H0_band,
                   cls_of_chan=cls_of_chan, terms=terms, dt=dt, rtol=rtol, max_iter=max_iter, n_steps=n_steps,
                   g_of_t=g_of_t, c0=c0, seed=seed,
                   meta=dict(kappas=kappas, chans=chans, dense=dense, c=c, l_max=l_max, kappa_max=kappa_max, l_of_term=l_of_term,
                             c_alpha=c_alpha, t_pulse=t_pulse, e0=e0, omega=omega))


def set_ground_state(p: Problem) -> Problem:
    """c0 = the lowest positive-branch eigenstate of the kappa = -1 block (1s1/2, mu = +1/2), S-normalised."""
    import scipy.linalg as sla
    S, H = p.meta["dense"][-1]
    E, V = sla.eigh(H, S)
    j = int(np.nonzero(E > -p.meta["c"] ** 2)[0][0])
    a = p.meta["chans"].index((-1, 0.5))
    p.c0[:] = 0.0
    p.c0[a * p.n_rad:(a + 1) * p.n_rad] = V[:, j]
    return p
