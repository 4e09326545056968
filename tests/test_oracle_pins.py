"""Pins for the oracle: each test checks oracle/ against something that is
*not* the oracle -- dense LAPACK solves, closed forms, invariants, textbook special cases.
CPU only."""
import math
import os

import numpy as np
import pytest
import scipy.linalg as sla
import scipy.sparse as sp

from oracle import tdde_oracle as orc
from tdde_inputs import band_to_dense, make_config, make_hydrogen, make_synthetic

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- dense helpers (numpy only)
def csr_to_dense(term, n_ang):
    A = np.zeros((n_ang, n_ang), dtype=np.complex128)
    for a in range(n_ang):
        for k in range(term.A_rowptr[a], term.A_rowptr[a + 1]):
            A[a, term.A_col[k]] += term.A_val[k]
    return A


def dense_operators(p):
    """S, H0, [K_L] as dense matrices built with numpy.kron -- independent of oracle.assemble."""
    n = p.n
    S = np.zeros((n, n), dtype=np.complex128)
    H0 = np.zeros((n, n), dtype=np.complex128)
    for k in range(p.n_cls):
        sel = np.diag((p.cls_of_chan == k).astype(np.float64))
        S += np.kron(sel, band_to_dense(p.S_band[k]))
        H0 += np.kron(sel, band_to_dense(p.H0_band[k]))
    K = [np.kron(csr_to_dense(t, p.n_ang), band_to_dense(t.R_band)) for t in p.terms]
    return S, H0, K


def dense_step(S, H0, K, g, dt, c):
    H = H0 + sum(gl * KL for gl, KL in zip(g, K))
    A = S + 0.5j * dt * H
    B = S - 0.5j * dt * H
    return np.linalg.solve(A, B @ c)


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.fixture(scope="module")
def tiny():
    p = make_config("tiny")
    return p, orc.assemble(p), orc.factor_precond(p)


@pytest.fixture(scope="module")
def tiny_stress():
    p = make_config("tiny", phase=math.pi / 2, e0=5.0)
    return p, orc.assemble(p), orc.factor_precond(p)


@pytest.fixture(scope="module")
def tiny_dense(tiny):
    return dense_operators(tiny[0])


@pytest.fixture(scope="module")
def hyd():
    p = make_hydrogen()
    return p


# ----------------------------------------------------------------------------- P9 Kronecker / assembly
def test_p9_csr_equals_scipy_kron(tiny):
    p, ops, _ = tiny
    for t, KL in zip(p.terms, ops.K):
        A = sp.csr_matrix((t.A_val, t.A_col, t.A_rowptr), shape=(p.n_ang, p.n_ang))
        R = sp.csr_matrix(band_to_dense(t.R_band))
        ref = sp.kron(A, R, format="csr")
        assert abs(KL - ref).max() < 1e-15


def test_p9_dense_kron_equals_csr(tiny, tiny_dense):
    p, ops, _ = tiny
    S, H0, K = tiny_dense
    assert np.abs(ops.S.toarray() - S).max() == 0.0
    assert np.abs(ops.H0.toarray() - H0).max() == 0.0
    for KL, Kd in zip(ops.K, K):
        assert np.abs(KL.toarray() - Kd).max() < 1e-15


def test_p9_vec_identity_and_linearity(tiny):
    p, ops, _ = tiny
    rng = np.random.default_rng(5)
    x = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    X = x.reshape(p.n_ang, p.n_rad)
    for t, KL in zip(p.terms, ops.K):
        ref = csr_to_dense(t, p.n_ang) @ X @ band_to_dense(t.R_band).T      # (A (x) R) vec(X) = vec(A X R^T)
        assert rel(KL @ x, ref.reshape(-1)) < 1e-13
    g1 = np.array([0.3, -0.7, 1.1])
    g2 = np.array([-0.2, 0.4, 0.9])
    y1 = orc.apply(ops, 1.0, 1j, g1, x)
    y2 = orc.apply(ops, 1.0, 1j, g2, x)
    y12 = orc.apply(ops, 2.0, 2j, 0.5 * (g1 + g2), x)
    assert rel(y1 + y2, y12) < 1e-13


def test_p9_hermiticity(tiny):
    p, ops, _ = tiny
    rng = np.random.default_rng(6)
    u = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    v = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    g = np.array([0.3, -0.7, 1.1])
    a = np.vdot(u, orc.apply_H(ops, g, v))
    b = np.conj(np.vdot(v, orc.apply_H(ops, g, u)))
    assert abs(a - b) / abs(a) < 1e-13
    assert abs(np.vdot(u, ops.S @ v) - np.conj(np.vdot(v, ops.S @ u))) < 1e-12


def test_block_structure(tiny):
    """H0 and S are block-diagonal over channels and depend on the class only."""
    p, ops, _ = tiny
    n_rad = p.n_rad
    coo = ops.H0.tocoo()
    assert np.all(coo.row // n_rad == coo.col // n_rad)
    a, b = 2, 3          # same class (cls 1)
    assert p.cls_of_chan[a] == p.cls_of_chan[b]
    Ha = ops.H0[a * n_rad:(a + 1) * n_rad, a * n_rad:(a + 1) * n_rad]
    Hb = ops.H0[b * n_rad:(b + 1) * n_rad, b * n_rad:(b + 1) * n_rad]
    assert abs(Ha - Hb).max() == 0.0


def test_p10_sampled_rows_match_csr(tiny_stress, hyd):
    p, ops, _ = tiny_stress
    rng = np.random.default_rng(7)
    x = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    g = np.array([0.3, -0.7, 1.1])
    alpha, beta = 0.7 - 0.2j, 0.1 + 0.9j
    y = orc.apply(ops, alpha, beta, g, x)
    chan = rng.integers(0, p.n_ang, 200)
    rad = rng.integers(0, p.n_rad, 200)
    chan[:4], rad[:4] = [0, 0, p.n_ang - 1, p.n_ang - 1], [0, p.n_rad - 1, 0, p.n_rad - 1]
    ys = orc.apply_rows_sampled(p, alpha, beta, g, x, chan, rad)
    ref = y[chan * p.n_rad + rad]
    assert np.max(np.abs(ys - ref)) / np.max(np.abs(ref)) < 1e-13
    # non-banded A (hydrogen)
    ph = hyd
    opsh = orc.assemble(ph)
    xh = rng.standard_normal(ph.n) + 1j * rng.standard_normal(ph.n)
    gh = np.full(ph.n_terms, 0.37)
    yh = orc.apply(opsh, 1.0, 0.5j, gh, xh)
    chan = rng.integers(0, ph.n_ang, 100)
    rad = rng.integers(0, ph.n_rad, 100)
    ys = orc.apply_rows_sampled(ph, 1.0, 0.5j, gh, xh, chan, rad)
    ref = yh[chan * ph.n_rad + rad]
    assert np.max(np.abs(ys - ref)) / np.max(np.abs(ref)) < 1e-12


def test_p10_apply_panels_vs_dense_kron_and_csr(tiny_stress, hyd):
    """The panel-streamed full-vector apply (used where the CSR cannot be held) against dense numpy.kron
    operators (independent of the oracle) on Tiny, and against the CSR apply on the non-banded hydrogen A and on a
    ragged shape; panel sizes that do not divide N_ang, a panel of one channel and one panel for everything."""
    p, ops, _ = tiny_stress
    S, H0, K = dense_operators(p)
    rng = np.random.default_rng(17)
    x = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    g = np.array([0.3, -0.7, 1.1])
    alpha, beta = 0.7 - 0.2j, 0.1 + 0.9j
    ref = alpha * (S @ x) + beta * ((H0 + sum(gl * KL for gl, KL in zip(g, K))) @ x)
    for panel in (1, 5, 16, 1000):
        assert rel(orc.apply_panels(p, alpha, beta, g, x, panel=panel), ref) < 1e-13, panel
    # a zero g_L skips the term; g = 0 leaves the block part
    g0 = np.array([0.0, 0.5, 0.0])
    assert rel(orc.apply_panels(p, 1.0, 0.5j, g0, x, panel=7), S @ x + 0.5j * ((H0 + 0.5 * K[1]) @ x)) < 1e-13
    ph = hyd
    opsh = orc.assemble(ph)
    xh = rng.standard_normal(ph.n) + 1j * rng.standard_normal(ph.n)
    gh = np.linspace(0.2, 0.9, ph.n_terms)
    assert rel(orc.apply_panels(ph, 1.0, 0.5j, gh, xh, panel=9), orc.apply(opsh, 1.0, 0.5j, gh, xh)) < 1e-13
    pr = make_synthetic(n_ang=37, n_r=11, bandwidth=13, n_terms=5, dt=0.01, n_steps=1, rtol=1e-10, seed=4)
    xr = rng.standard_normal(pr.n) + 1j * rng.standard_normal(pr.n)
    gr = np.linspace(-1.0, 1.0, 5)
    assert rel(orc.apply_panels(pr, 0.3, 1.0 - 2.0j, gr, xr, panel=16), orc.apply(orc.assemble(pr), 0.3, 1.0 - 2.0j, gr, xr)) < 1e-13


def test_cn_step_panels_vs_dense_lu(tiny_stress, tiny_dense):
    """The matrix-free CN step (cn_step_panels) solves the same dense system as P1."""
    p, ops, fact = tiny_stress
    S, H0, K = tiny_dense
    g = p.g_mid(1)
    c1, info = orc.cn_step_panels(p, fact, p.c0, g, p.dt, p.rtol, p.max_iter, panel=5)
    assert info.status == "ok" and info.half_iters >= 2
    assert rel(c1, dense_step(S, H0, K, g, p.dt, p.c0)) < 1e-10


# ----------------------------------------------------------------------------- P8 preconditioner
def test_p8_precond_vs_dense_solve(tiny):
    p, ops, fact = tiny
    rng = np.random.default_rng(8)
    x = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    y = orc.apply_precond(fact, x)
    tau = 0.5 * p.dt
    for a in (0, 3, 7, 15):
        k = p.cls_of_chan[a]
        M = band_to_dense(p.S_band[k]) + 1j * tau * band_to_dense(p.H0_band[k])
        ref = np.linalg.solve(M, x[a * p.n_rad:(a + 1) * p.n_rad])
        assert rel(y[a * p.n_rad:(a + 1) * p.n_rad], ref) < 1e-13
    # M (M^-1 x) = x through the assembled operators with g = 0
    back = orc.apply(ops, 1.0, 1j * tau, np.zeros(p.n_terms), y)
    assert rel(back, x) < 1e-13


def test_nopivot_lu_is_safe():
    """Reading R5b / SURVEY C5: the Hermitian part of M_k is S_k > 0, so LU without pivoting exists;
    its solve agrees with the pivoted LAPACK result at rounding level."""
    p = make_config("tiny")
    tau = 0.5 * p.dt
    M = band_to_dense(p.S_band[0]) + 1j * tau * band_to_dense(p.H0_band[0])
    n = M.shape[0]
    LU = M.copy()
    for j in range(n - 1):               # textbook Doolittle elimination, no pivoting
        LU[j + 1:, j] /= LU[j, j]
        LU[j + 1:, j + 1:] -= np.outer(LU[j + 1:, j], LU[j, j + 1:])
    L = np.tril(LU, -1) + np.eye(n)
    U = np.triu(LU)
    assert np.abs(L @ U - M).max() < 1e-14
    w = p.w0
    ii, jj = np.indices(M.shape)
    assert np.abs(LU[np.abs(ii - jj) > w]).max() == 0.0          # no fill outside the band
    assert np.min(np.abs(np.diag(U))) > 0.3


# ----------------------------------------------------------------------------- BiCGSTAB itself
def test_bicgstab_small_dense_system():
    rng = np.random.default_rng(9)
    n = 60
    A = np.eye(n) * 4 + (rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))) * 0.3
    b = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    ref = np.linalg.solve(A, b)
    Mdiag = np.diag(A).copy()
    for M_solve in (lambda u: u.copy(), lambda u: u / Mdiag):
        x, info = orc.bicgstab(lambda u: A @ u, M_solve, b, np.zeros(n, complex), 1e-13, 200)
        assert info.converged and info.status == "ok"
        assert rel(x, ref) < 1e-11
        assert np.linalg.norm(b - A @ x) <= 1.01e-13 * np.linalg.norm(b) * 5


def test_bicgstab_trace_residual_identity(tiny_stress):
    """Along a forced trace the recursively updated r equals b - A x (to rounding) and
    s = r_prev - alpha v -- catches sign/ordering slips in the update formulas."""
    p, ops, fact = tiny_stress
    g = p.g_mid(0)
    tau = 0.5 * p.dt
    H = orc.hamiltonian_csr(ops, g)
    A = (ops.S + 1j * tau * H).tocsr()
    b = (ops.S - 1j * tau * H) @ p.c0
    x, info = orc.cn_step(ops, fact, p.c0, g, p.dt, p.rtol, p.max_iter, force_iters=4, keep_trace=True)
    assert len(info.trace) == 4 and info.half_iters == 8
    nb = np.linalg.norm(b)
    for it in info.trace:
        assert np.linalg.norm(it["r"] - (b - A @ it["x"])) / nb < 1e-13
        assert np.linalg.norm(A @ it["y"] - it["v"]) / np.linalg.norm(it["v"]) < 1e-13


def test_exact_precond_converges_in_half_step():
    """g = 0 => M^-1 A = I => s = 0 after the first half step (reading R11)."""
    p = make_config("tiny", e0=0.0)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x, info = orc.cn_step(ops, fact, p.c0, p.g_mid(0), p.dt, p.rtol, p.max_iter)
    assert info.half_iters == 1 and info.converged


# ----------------------------------------------------------------------------- P1 dense LU
@pytest.mark.parametrize("which", ["tiny", "tiny_stress"])
def test_p1_step_vs_dense_lu(which, tiny, tiny_stress, tiny_dense):
    p, ops, fact = tiny if which == "tiny" else tiny_stress
    S, H0, K = tiny_dense
    c_ref = p.c0.copy()
    c_orc = p.c0.copy()
    for s in range(p.n_steps):
        g = p.g_mid(s)
        c_ref = dense_step(S, H0, K, g, p.dt, c_ref)
        c_orc, info = orc.cn_step(ops, fact, c_orc, g, p.dt, p.rtol, p.max_iter)
        assert info.status == "ok"
    assert rel(c_orc, c_ref) < 1e-10
    c_prop, infos = orc.propagate(p, ops, fact, p.c0, p.n_steps)
    assert rel(c_prop, c_ref) < 1e-10
    c_sp, _ = orc.propagate(p, ops, fact, p.c0, p.n_steps, assembled=False)
    assert rel(c_sp, c_ref) < 1e-10
    if which == "tiny_stress":
        assert max(i.half_iters for i in infos) >= 4          # the stress run really iterates


# ----------------------------------------------------------------------------- P2 S-norm conservation
@pytest.mark.parametrize("which", ["tiny", "tiny_stress"])
def test_p2_s_norm_conserved(which, tiny, tiny_stress):
    p, ops, fact = tiny if which == "tiny" else tiny_stress
    n0 = orc.s_norm_sq(ops, p.c0)
    assert abs(n0 - 1.0) < 1e-12
    c, infos = orc.propagate(p, ops, fact, p.c0, p.n_steps)
    assert abs(orc.s_norm_sq(ops, c) - n0) <= 10 * p.n_steps * p.rtol
    assert rel(c, p.c0) > 1e-6                                   # the state actually moved


def test_s_norm_is_quadratic_form(tiny, tiny_dense):
    p, ops, _ = tiny
    S = tiny_dense[0]
    assert abs(orc.s_norm_sq(ops, p.c0) - np.real(np.conj(p.c0) @ S @ p.c0)) < 1e-13


# ----------------------------------------------------------------------------- P3 eigenstate phase
def test_p3_eigenstate_phase_synthetic():
    p = make_config("tiny", e0=0.0)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    a = 5
    k = p.cls_of_chan[a]
    Hk, Sk = band_to_dense(p.H0_band[k]), band_to_dense(p.S_band[k])
    E, V = sla.eigh(Hk, Sk)
    j = 17
    c0 = np.zeros(p.n, dtype=np.complex128)
    c0[a * p.n_rad:(a + 1) * p.n_rad] = V[:, j]
    tau = 0.5 * p.dt
    N = 10
    c, infos = orc.propagate(p, ops, fact, c0, N)
    phase = ((1 - 1j * tau * E[j]) / (1 + 1j * tau * E[j])) ** N
    assert rel(c, phase * c0) < 1e-9
    assert all(i.half_iters == 1 for i in infos)


def test_p3_p5_hydrogen_1s_stationary(hyd):
    p = make_hydrogen(field=False, n_steps=20)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    S, H = p.meta["dense"][-1]
    E, V = sla.eigh(H, S)
    c2 = p.meta["c"] ** 2
    j = int(np.nonzero(E > -c2)[0][0])
    c0 = np.zeros(p.n, dtype=np.complex128)
    a = 1                                    # kappa = -1, mu = +1/2
    assert p.meta["chans"][a] == (-1, 0.5)
    c0[a * p.n_rad:(a + 1) * p.n_rad] = V[:, j]
    tau = 0.5 * p.dt
    c, infos = orc.propagate(p, ops, fact, c0, p.n_steps)
    phase = ((1 - 1j * tau * E[j]) / (1 + 1j * tau * E[j])) ** p.n_steps
    assert rel(c, phase * c0) < 1e-9
    assert all(i.half_iters == 1 for i in infos)


# ----------------------------------------------------------------------------- P4 time reversal
def test_p4_time_reversal(tiny_stress):
    p, ops, fact = tiny_stress
    g = p.g_mid(3)
    c1, i1 = orc.cn_step(ops, fact, p.c0, g, p.dt, p.rtol, p.max_iter)
    fact_m = orc.factor_precond(p, dt=-p.dt)
    c2, i2 = orc.cn_step(ops, fact_m, c1, g, -p.dt, p.rtol, p.max_iter)
    assert i1.status == "ok" and i2.status == "ok"
    assert rel(c2, p.c0) < 10 * p.rtol * 10


# ----------------------------------------------------------------------------- midpoint rule / order
def test_midpoint_sampling_gives_second_order():
    """With g sampled at t_{n+1/2} (reading R1) the CN propagation of a time-dependent H is second
    order in dt; sampling at t_n or t_{n+1} would be first order.  Reference: fine-step dense
    exponential midpoint propagation (scipy.linalg.expm)."""
    def build(dt, n_steps):
        return make_synthetic(n_ang=4, n_r=6, bandwidth=5, n_terms=2, dt=dt, n_steps=n_steps, rtol=1e-14,
                              seed=11, e0=2.0, omega=3.0, phase=0.3, name="order")
    T = 0.4
    p_ref = build(T / 4096, 4096)
    S, H0, K = dense_operators(p_ref)
    Sinv = np.linalg.inv(S)
    c = p_ref.c0.copy()
    for s in range(4096):
        g = p_ref.g_mid(s)
        H = H0 + sum(gl * KL for gl, KL in zip(g, K))
        c = sla.expm(-1j * p_ref.dt * (Sinv @ H)) @ c
    errs = []
    for n_steps in (16, 32, 64):
        p = build(T / n_steps, n_steps)
        ops, fact = orc.assemble(p), orc.factor_precond(p)
        cc, _ = orc.propagate(p, ops, fact, p.c0, n_steps)
        errs.append(rel(cc, c))
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5, errs


# ----------------------------------------------------------------------------- P5 / P6 hydrogen spectrum
def read_golden_levels():
    out = {}
    with open(os.path.join(GOLD, "hydrogen_energies.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            lab, n, k, e = line.split()
            out[lab] = (int(n), int(k), float(e))
    return out


def test_golden_1s_is_north_star_closed_form():
    c = 137.035999084
    lv = read_golden_levels()
    assert abs(lv["1s1/2"][2] - c * c * (math.sqrt(1 - (1 / c) ** 2) - 1)) < 1e-11


def test_p5_p6_hydrogen_levels(hyd):
    lv = read_golden_levels()
    c2 = hyd.meta["c"] ** 2
    n_r = hyd.meta["n_r"]
    by_kappa = {}
    for lab, (n, k, e) in lv.items():
        by_kappa.setdefault(k, []).append((n, e))
    for kap, (S, H) in hyd.meta["dense"].items():
        E = sla.eigh(H, S, eigvals_only=True)
        assert int(np.sum(E < -c2)) == n_r                         # P6: no spurious states
        pos = E[E > -c2]
        for n, e in sorted(by_kappa.get(kap, [])):
            idx = n - (abs(kap) if kap < 0 else kap + 1)           # radial quantum number
            assert abs(pos[idx] - e) < 1e-9, (kap, n, pos[idx], e)


# ----------------------------------------------------------------------------- P7 angular factors
def cg_spinor(kappa, mu):
    """(coefficient of Y_{l,mu-1/2} spin-up, coefficient of Y_{l,mu+1/2} spin-down) from the
    Clebsch-Gordan table for l (x) 1/2 (Eq. 8)."""
    l = kappa if kappa > 0 else -kappa - 1
    if kappa < 0:       # j = l + 1/2
        return l, math.sqrt((l + 0.5 + mu) / (2 * l + 1)), math.sqrt((l + 0.5 - mu) / (2 * l + 1))
    return l, -math.sqrt((l + 0.5 - mu) / (2 * l + 1)), math.sqrt((l + 0.5 + mu) / (2 * l + 1))


def test_p7_sigma_z_elements():
    from tdde_inputs.hydrogen import sigma_z_element
    assert abs(sigma_z_element(-1, -1, 0.5) - 1.0) < 1e-15
    assert abs(sigma_z_element(1, 1, 0.5) + 1.0 / 3.0) < 1e-15
    for k1 in range(-5, 6):
        if k1 == 0:
            continue
        j1 = abs(k1) - 0.5
        mu = -j1
        while mu <= j1 + 1e-9:
            tot = 0.0
            for k2 in range(-7, 8):
                if k2 == 0 or abs(mu) > abs(k2) - 0.5 + 1e-9:
                    continue
                l1, u1, d1 = cg_spinor(k1, mu)
                l2, u2, d2 = cg_spinor(k2, mu)
                direct = (u1 * u2 - d1 * d2) if l1 == l2 else 0.0       # <chi1|sigma_z|chi2>, Y_lm orthonormal
                assert abs(sigma_z_element(k1, k2, mu) - direct) < 1e-14
                tot += sigma_z_element(k1, k2, mu) ** 2
            assert abs(tot - 1.0) < 1e-14                               # sigma_z^2 = 1
            mu += 1.0


def test_hydrogen_interaction_hermitian_and_velocity_form(hyd):
    """The assembled dipole operator is Hermitian, and its 1s -> 2p matrix elements reproduce the
    velocity-form identity <f|c alpha_z|i> = i (E_f - E_i) <f|z|i> with the non-relativistic
    <2p0|z|1s> = 128 sqrt(2)/243 (relativistic corrections are O(alpha^2))."""
    p = hyd
    ops = orc.assemble(p)
    D = sum(ops.K)                           # g_L = 1 for every term: -c alpha_z
    assert abs(D - D.getH()).max() < 1e-9 * abs(D).max()
    c2 = p.meta["c"] ** 2
    n_rad = p.n_rad
    chans = p.meta["chans"]

    def state(kappa, mu, level):
        S, H = p.meta["dense"][kappa]
        E, V = sla.eigh(H, S)
        j = int(np.nonzero(E > -c2)[0][0]) + level
        a = chans.index((kappa, mu))
        v = np.zeros(p.n, dtype=np.complex128)
        v[a * n_rad:(a + 1) * n_rad] = V[:, j]
        return E[j], v

    E1s, v1s = state(-1, 0.5, 0)
    tot = 0.0
    for kap in (1, -2):
        E2p, v2p = state(kap, 0.5, 0)
        assert abs(E2p + 0.125) < 1e-5
        tot += abs(np.vdot(v2p, D @ v1s)) ** 2
    ref = (0.375 * 128 * math.sqrt(2) / 243) ** 2
    assert abs(tot - ref) / ref < 2e-4


def test_hydrogen_norm_conserved_under_field():
    p = make_hydrogen(n_steps=25, t_offset=150.0, rtol=1e-12)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    assert abs(p.g_mid(0)[0]) > 0.3                  # mid-pulse: A(t) ~ E0/omega
    S, H = p.meta["dense"][-1]
    E, V = sla.eigh(H, S)
    j = int(np.nonzero(E > -p.meta["c"] ** 2)[0][0])
    c0 = np.zeros(p.n, dtype=np.complex128)
    c0[p.n_rad:2 * p.n_rad] = V[:, j]
    n0 = orc.s_norm_sq(ops, c0)
    assert abs(n0 - 1.0) < 1e-10
    c, infos = orc.propagate(p, ops, fact, c0, p.n_steps)
    assert all(i.status == "ok" for i in infos)
    assert abs(orc.s_norm_sq(ops, c) - n0) < 10 * p.n_steps * p.rtol * 10
    leaked = 1.0 - abs(np.vdot(c0, ops.S @ c)) ** 2
    assert leaked > 1e-6                              # the field really couples channels


# ----------------------------------------------------------------------------- NEXT-1: paper-shaped angular operators (Eq. 17-18, 27-30)
def test_clebsch_gordan_and_3j_vs_sympy_and_orthogonality():
    """Racah-formula Clebsch-Gordan coefficients and 3j symbols of tdde_inputs.nondipole against sympy's exact values, and the
    orthogonality sums every such table obeys."""
    from sympy import N, Rational as Rq
    from sympy.physics.wigner import clebsch_gordan as scg, wigner_3j as s3j
    from tdde_inputs import nondipole as nd
    for tj1, tj2 in [(2, 1), (6, 1), (3, 2), (5, 4), (20, 1), (31, 1)]:
        for tJ in range(abs(tj1 - tj2), tj1 + tj2 + 1, 2):
            for tm1 in range(-tj1, tj1 + 1, 2):
                for tm2 in range(-tj2, tj2 + 1, 2):
                    ref = float(N(scg(Rq(tj1, 2), Rq(tj2, 2), Rq(tJ, 2), Rq(tm1, 2), Rq(tm2, 2), Rq(tm1 + tm2, 2)), 30))
                    assert abs(nd.clebsch_gordan(tj1, tm1, tj2, tm2, tJ, tm1 + tm2) - ref) < 1e-13
    for l1, l2, l3 in [(2, 1, 1), (4, 2, 2), (7, 3, 4), (10, 10, 0), (12, 2, 14)]:
        tot = 0.0
        for m1 in range(-l1, l1 + 1):
            for m2 in range(-l2, l2 + 1):
                v = nd.wigner_3j(l1, l2, l3, m1, m2, -m1 - m2)
                if abs(m1 + m2) <= l3:
                    assert abs(v - float(N(s3j(l1, l2, l3, m1, m2, -m1 - m2), 30))) < 1e-13
                tot += v * v
        assert abs(tot - 1.0) < 1e-13                      # sum over m1, m2, m3 of (3j)^2 = 1
    # unitarity of the coupling: sum_{m1} <j1 m1 j2 M-m1 | J M> <j1 m1 j2 M-m1 | J' M> = delta_{J J'}
    tj1, tj2, tM = 8, 3, 3
    Js = list(range(abs(tj1 - tj2), tj1 + tj2 + 1, 2))
    G = np.array([[sum(nd.clebsch_gordan(tj1, tm1, tj2, tM - tm1, a, tM) * nd.clebsch_gordan(tj1, tm1, tj2, tM - tm1, b, tM)
                       for tm1 in range(-tj1, tj1 + 1, 2)) for b in Js] for a in Js])
    assert np.max(np.abs(G - np.eye(len(Js)))) < 1e-13


def test_h_theta_by_quadrature_on_the_sphere():
    """(H^theta_l)_{k'k mu'mu} = 4 pi Y_l0(z) <X_{-k',mu'}| sigma_x Y_l0 |X_{k,mu}> (Eq. 18) by brute force: spinor
    components from sympy's Clebsch-Gordan coefficients and scipy's spherical harmonics, integrated with Gauss-Legendre x
    uniform quadrature over the sphere -- no 3j symbol, no code of the generator."""
    from scipy.special import sph_harm_y
    from sympy import N, Rational as Rq
    from sympy.physics.wigner import clebsch_gordan as scg
    from tdde_inputs import nondipole as nd
    from tdde_inputs.hydrogen import l_of_kappa
    xg, wg = np.polynomial.legendre.leggauss(24)
    phi = 2 * np.pi * np.arange(48) / 48
    TH, PH = np.meshgrid(np.arccos(xg), phi, indexing="ij")
    Wt = np.outer(wg, np.full(48, 2 * np.pi / 48))

    def spinor(kappa, mu):                                  # (up, down) components on the grid
        l, j = l_of_kappa(kappa), abs(kappa) - 0.5
        comps = []
        for ms in (0.5, -0.5):
            m = mu - ms
            if abs(m) > l:
                comps.append(np.zeros_like(TH, dtype=complex))
                continue
            cg = float(N(scg(l, Rq(1, 2), Rq(int(2 * j), 2), int(round(m)), Rq(int(2 * ms), 2), Rq(int(round(2 * mu)), 2)), 20))
            comps.append(cg * sph_harm_y(l, int(round(m)), TH, PH))
        return comps

    rng = np.random.default_rng(0)
    cases = [(0, 1, 1, 0.5, -0.5), (0, -1, -1, -0.5, 0.5), (1, -1, -2, 0.5, 1.5), (1, 2, 1, -0.5, 0.5), (2, -2, 3, 1.5, 2.5), (2, 3, -3, -1.5, -0.5),
             (3, -4, 2, 2.5, 1.5), (1, 1, 1, 0.5, -0.5), (2, -1, -1, 0.5, -0.5)]
    for l, kp, k, mup, mu in cases:
        bu, bd = spinor(-kp, mup)
        ku, kd = spinor(k, mu)
        yl0 = sph_harm_y(l, 0, TH, PH)
        val = np.sum(Wt * yl0 * (np.conj(bu) * kd + np.conj(bd) * ku))          # sigma_x swaps the components
        ref = 4 * np.pi * np.sqrt((2 * l + 1) / (4 * np.pi)) * val
        got = nd.h_theta_element(l, kp, k, int(round(2 * mup)), int(round(2 * mu)))
        assert abs(ref.imag) < 1e-12 and abs(got - ref.real) < 1e-12, (l, kp, k, mup, mu, got, ref)


def test_h_theta_selection_rules_sum_rule_and_growth():
    """Zero pattern = {mu = mu' +- 1} and the l-triangle / parity rule (Eq. 29-30); sigma_x^2 = 1 gives the sum
    rule sum_{k mu} (H^theta_0)^2 = 1 per row whose partners all lie inside kappa_max; the number of non-zeros of the coupling
    pattern grows like kappa_max^2 at fixed l_max (Fig. 2)."""
    from tdde_inputs import nondipole as nd
    from tdde_inputs.hydrogen import channel_list, l_of_kappa
    _, chans, _ = channel_list(5)
    for l in range(0, 4):
        H = nd.h_theta(l, chans)
        for i, (kp, mup) in enumerate(chans):
            for j, (k, mu) in enumerate(chans):
                allowed = abs(mu - mup) == 1.0 and nd.triangle_allows(l, kp, k)
                full = nd.h_theta_element(l, kp, k, int(round(2 * mup)), int(round(2 * mu)))       # without the mu shortcut
                assert abs(full - H[i, j]) < 1e-15
                if not allowed:
                    assert H[i, j] == 0.0 or abs(H[i, j]) < 1e-14, (l, kp, k, mup, mu)
        assert np.count_nonzero(np.abs(H) > 1e-12) > 0
    H0 = nd.h_theta(0, chans)
    inner = [i for i, (kp, _) in enumerate(chans) if abs(kp) <= 3]          # sigma_x X_{k,mu} only reaches |kappa| + 1
    assert np.max(np.abs(np.sum(H0[inner] ** 2, axis=1) - 1.0)) < 1e-13
    # growth: the pattern is exactly the selection rules (just verified entry by entry), so count those for larger kappa_max
    def rule_count(kmax, lmax):
        kaps = [s * m for m in range(1, kmax + 1) for s in (-1, 1)]
        tot = 0
        for kp in kaps:
            for k in kaps:
                if not any(nd.triangle_allows(l, kp, k) for l in range(lmax + 1)):
                    continue
                # the spherical harmonics of both spinor components must exist: |m| <= l on each side, m = mu' + ms = mu - ms
                lb, lk, jp, j = l_of_kappa(-kp), l_of_kappa(k), abs(kp) - 0.5, abs(k) - 0.5
                for mup in np.arange(-jp, jp + 1):
                    for ms in (-0.5, 0.5):
                        tot += abs(mup + 2 * ms) <= j and abs(mup + ms) <= min(lb, lk)
        return tot
    _, ch, _ = channel_list(4)
    pat = np.zeros((len(ch), len(ch)), dtype=bool)
    for l in range(3):
        pat |= np.abs(nd.h_theta(l, ch)) > 1e-13
    assert int(pat.sum()) == rule_count(4, 2)
    counts = [rule_count(kmax, 2) for kmax in (8, 16, 32, 64)]
    ratios = [counts[i + 1] / counts[i] for i in range(3)]
    assert all(3.7 < r < 4.7 for r in ratios) and abs(ratios[2] - 4.0) < 0.15, (counts, ratios)


def test_nondipole_operator_hermitian_and_norm_conserving():
    """Eq. 17: each bracket alone is not Hermitian, their sum is; the oracle's CN step then conserves the
    S-norm under the field.  The panel-streamed apply agrees with the CSR apply on this non-banded, 24-term operator."""
    from tdde_inputs import nondipole as nd
    p = nd.make_nondipole(kappa_max=2, l_max=2, n_r=9)
    g = p.g_mid(40)
    assert np.all(g != 0.0) and p.n_terms == 24
    HI = sum(gl * np.kron(csr_to_dense(t, p.n_ang), band_to_dense(t.R_band)) for gl, t in zip(g, p.terms))
    assert np.linalg.norm(HI - HI.conj().T) <= 1e-13 * np.linalg.norm(HI)
    first = sum(gl * np.kron(csr_to_dense(t, p.n_ang), band_to_dense(t.R_band)) for gl, t in zip(g[0::2], p.terms[0::2]))
    assert np.linalg.norm(first - first.conj().T) > 1e-3 * np.linalg.norm(first)
    p = nd.set_ground_state(nd.make_nondipole(kappa_max=3, l_max=2, n_r=12))
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c, infos = orc.propagate(p, ops, fact, p.c0, 4, first_step=60)
    assert all(i.status == "ok" for i in infos) and max(i.half_iters for i in infos) >= 2
    assert abs(orc.s_norm_sq(ops, c) - orc.s_norm_sq(ops, p.c0)) <= 40 * p.rtol
    x = np.random.default_rng(3).standard_normal(2 * p.n).view(np.complex128)
    gg = p.g_mid(60)
    assert rel(orc.apply_panels(p, 1.0, 0.5j * p.dt, gg, x, panel=7), orc.apply(ops, 1.0, 0.5j * p.dt, gg, x)) < 1e-13


# ----------------------------------------------------------------------------- NEXT-4: projection on field-free eigenstates (Eq. 33)
def _eigenbasis(p):
    """Eigenvectors of every kappa-class pencil (H0_k, S_k) by LAPACK (scipy.linalg.eigh), S-orthonormal: V[k, e, :]."""
    V = np.zeros((p.n_cls, p.n_rad, p.n_rad), dtype=np.complex128)
    E = np.zeros((p.n_cls, p.n_rad))
    for k in range(p.n_cls):
        E[k], vec = sla.eigh(band_to_dense(p.H0_band[k]), band_to_dense(p.S_band[k]))
        V[k] = vec.T
    return E, V


def test_projection_on_eigenstates_delta_and_completeness():
    """oracle.project: an eigenstate projects onto itself only (S-orthonormality of the generalised eigenvectors), and over the
    full eigenbasis of a channel the probabilities add up to that channel's share of the S-norm (completeness)."""
    p = make_synthetic(n_ang=9, n_r=12, bandwidth=7, n_terms=0, dt=0.01, n_steps=1, rtol=1e-10, seed=2)
    E, V = _eigenbasis(p)
    c = np.zeros(p.n, dtype=np.complex128)
    a0, e0 = 5, 7
    c[a0 * p.n_rad:(a0 + 1) * p.n_rad] = (0.6 + 0.8j) * V[p.cls_of_chan[a0], e0]
    P = orc.project(p, V, c)
    ref = np.zeros_like(P)
    ref[a0, e0] = 1.0
    assert np.max(np.abs(P - ref)) < 1e-12
    rng = np.random.default_rng(1)
    x = rng.standard_normal(2 * p.n).view(np.complex128)
    P = orc.project(p, V, x)
    ops = orc.assemble(p)
    X = x.reshape(p.n_ang, p.n_rad)
    per_chan = np.array([np.real(np.vdot(X[a], band_to_dense(p.S_band[p.cls_of_chan[a]]) @ X[a])) for a in range(p.n_ang)])
    assert np.max(np.abs(P.sum(axis=1) - per_chan)) < 1e-11 * per_chan.max()
    assert abs(P.sum() - orc.s_norm_sq(ops, x)) < 1e-11 * P.sum()


def test_oracle_eigenstates_match_closed_form_and_pencil(hyd):
    """oracle.eigenstates on the hydrogen blocks: the bound levels are the Sommerfeld closed form (golden file, P5), every pair
    satisfies H v = E S v, and the vectors are S-orthonormal."""
    p = hyd
    E, V = orc.eigenstates(p)
    c2 = p.meta["c"] ** 2
    levels = read_golden_levels()
    k1 = p.meta["kappas"].index(-1)
    pos = E[k1][E[k1] > -c2]
    assert abs(pos[0] - levels["1s1/2"][2]) < 1e-9 and abs(pos[1] - levels["2s1/2"][2]) < 1e-9
    k2 = p.meta["kappas"].index(-2)
    assert abs(E[k2][E[k2] > -c2][0] - levels["2p3/2"][2]) < 1e-9
    for k in (0, 3):
        S, H = band_to_dense(p.S_band[k]), band_to_dense(p.H0_band[k])
        R = H @ V[k].T - (S @ V[k].T) * E[k][None, :]
        assert np.linalg.norm(R) <= 1e-9 * np.linalg.norm(H)
        assert np.max(np.abs(V[k].conj() @ S @ V[k].T - np.eye(p.n_rad))) < 1e-9
