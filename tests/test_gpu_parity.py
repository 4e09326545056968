"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Tolerances (BASELINE.json north_star): relative L2 <= 1e-12 per operator apply, <= 1e-9 on the wavefunction
after a propagation.  Integer results (iteration counts) are compared exactly where both sides are far from
the tolerance edge, +-1 half-iteration otherwise ("parity unpinned" for counts).
"""
import numpy as np
import pytest

import tdde_inputs
from oracle import tdde_oracle as orc

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def make(name, **kw):
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_config(name, **kw) if isinstance(name, str) else name
    return p, Tdde(p)


def rand_vec(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(2 * n).view(np.complex128).copy()


# a reduced Medium: same structure as BASELINE configs[2] (w = 6, T = 5, offsets 1..L+1), sized for the oracle's CSR
SMALL_MED = dict(n_ang=100, n_r=150, bandwidth=13, n_terms=5, dt=0.005, n_steps=6, rtol=1e-10, seed=11)


@pytest.fixture(scope="module")
def tiny():
    p, prop = make("tiny")
    yield p, prop, orc.assemble(p), orc.factor_precond(p)
    prop.close()


@pytest.fixture(scope="module")
def tiny_stress():
    p, prop = make("tiny", phase=np.pi / 2, e0=5.0)
    yield p, prop, orc.assemble(p), orc.factor_precond(p)
    prop.close()


@pytest.fixture(scope="module")
def smallmed():
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(name="smallmed", phase=np.pi / 2, e0=2.0, **SMALL_MED)
    prop = Tdde(p)
    yield p, prop, orc.assemble(p), orc.factor_precond(p)
    prop.close()


@pytest.fixture(scope="module")
def hyd():
    from paper_2512_21697_b200 import Tdde
    import scipy.linalg as sla
    p = tdde_inputs.make_hydrogen()
    # c0 = the 1s1/2 (kappa = -1, mu = +1/2) eigenstate of the field-free block, S-normalised by eigh
    S, H = p.meta["dense"][-1]
    E, V = sla.eigh(H, S)
    j = int(np.nonzero(E > -p.meta["c"] ** 2)[0][0])
    a = p.meta["chans"].index((-1, 0.5))
    p.c0[a * p.n_rad:(a + 1) * p.n_rad] = V[:, j]
    prop = Tdde(p)
    yield p, prop, orc.assemble(p), orc.factor_precond(p)
    prop.close()


def test_paths_selected(tiny, smallmed, hyd):
    assert tiny[1].apply_path == "banded"
    assert smallmed[1].apply_path == "banded"
    assert hyd[1].apply_path == "staged"


@pytest.mark.parametrize("which", ["tiny", "smallmed", "hyd"])
def test_apply_parity(which, request):
    p, prop, ops, _ = request.getfixturevalue(which)
    x = rand_vec(p.n, 5)
    xd = prop.to_device(x)
    rng = np.random.default_rng(3)
    for alpha, beta, g in [(1.0, 0.5j * p.dt, p.g_mid(3)), (1.0, -0.5j * p.dt, rng.standard_normal(p.n_terms)),
                           (0.3 - 0.2j, 1.0 + 0.5j, rng.standard_normal(p.n_terms)), (1.0, 0.0, np.zeros(p.n_terms)),
                           (0.0, 1.0, np.ones(p.n_terms))]:
        y = prop.apply(alpha, beta, g, xd).cpu().numpy()
        y_ref = orc.apply(ops, alpha, beta, np.asarray(g, dtype=float), x)
        assert rel(y, y_ref) <= 1e-12, (which, alpha, beta)


def test_apply_ragged_shapes():
    """Channel counts that are not multiples of 32/128 and radial sizes that do not divide the segment length."""
    from paper_2512_21697_b200 import Tdde
    for n_ang, n_r, T, bw in [(1, 8, 1, 7), (2, 9, 2, 7), (33, 17, 2, 7), (130, 37, 5, 13), (257, 23, 7, 13), (40, 31, 7, 19)]:
        p = tdde_inputs.make_synthetic(n_ang=n_ang, n_r=n_r, bandwidth=bw, n_terms=T, dt=0.01, n_steps=1, rtol=1e-10,
                                       seed=n_ang, name="ragged")
        if n_ang <= T + 1:      # offsets beyond the matrix leave empty terms: must fall back to the generic path
            pass
        prop = Tdde(p)
        ops = orc.assemble(p)
        x = rand_vec(p.n, 1)
        g = np.linspace(0.5, 1.5, T)
        y = prop.apply(1.0, 0.25j, g, prop.to_device(x)).cpu().numpy()
        assert rel(y, orc.apply(ops, 1.0, 0.25j, g, x)) <= 1e-12, (n_ang, n_r, T, bw, prop.apply_path)
        z = prop.precond(prop.to_device(x)).cpu().numpy()
        assert rel(z, orc.apply_precond(orc.factor_precond(p), x)) <= 1e-12, (n_ang, n_r, T, bw)
        prop.close()


@pytest.mark.parametrize("which", ["tiny", "smallmed", "hyd"])
def test_precond_parity_p8(which, request):
    p, prop, ops, fact = request.getfixturevalue(which)
    x = rand_vec(p.n, 7)
    xd = prop.to_device(x)
    y = prop.precond(xd).cpu().numpy()
    assert rel(y, orc.apply_precond(fact, x)) <= 1e-12
    # M (M^-1 x) = x through tdde_apply with g = 0
    back = prop.apply(1.0, 0.5j * p.dt, np.zeros(p.n_terms), prop.to_device(y)).cpu().numpy()
    assert rel(back, x) <= 1e-12
    # in place
    prop.precond(xd, xd)
    assert rel(xd.cpu().numpy(), y) == 0.0


@pytest.mark.parametrize("which", ["tiny", "smallmed", "hyd"])
def test_norm_parity(which, request):
    p, prop, ops, _ = request.getfixturevalue(which)
    x = rand_vec(p.n, 9)
    assert abs(prop.norm(prop.to_device(x)) - orc.s_norm_sq(ops, x)) <= 1e-12 * orc.s_norm_sq(ops, x)


@pytest.mark.parametrize("which", ["tiny", "tiny_stress", "smallmed"])
def test_propagate_parity(which, request):
    p, prop, ops, fact = request.getfixturevalue(which)
    n_steps = min(p.n_steps, 10)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, n_steps)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(n_steps))
    assert st["steps"] == n_steps and st["status"] == 0
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    ref_half = sum(i.half_iters for i in infos)
    assert abs(st["half_iters"] - ref_half) <= n_steps, (st, ref_half)     # +-1 half-iteration per step at the edge
    assert st["rel_res"] <= p.rtol
    assert abs(prop.norm(c) - 1.0) <= 10 * n_steps * p.rtol                 # P2 on the GPU path


def test_step_equals_propagate_of_one(tiny_stress):
    p, prop, ops, fact = tiny_stress
    c1 = prop.to_device(p.c0)
    c2 = prop.to_device(p.c0)
    for s in range(3):
        prop.step(c1, p.g_mid(s))
    prop.propagate(c2, p.g_table(3))
    assert np.array_equal(c1.cpu().numpy(), c2.cpu().numpy())


def test_hydrogen_field_free_and_field(hyd):
    p, prop, ops, fact = hyd
    # field-free: exact preconditioner => the ||s|| exit at half-iteration 1 every step (C8-11, P3)
    c = prop.to_device(p.c0)
    g0 = np.zeros((5, p.n_terms))
    st = prop.propagate(c, g0)
    assert st["half_iters"] == 5 and st["steps"] == 5
    pz = tdde_inputs.Problem(**{**p.__dict__, "g_of_t": lambda t: np.zeros(p.n_terms)})
    c_ref, _ = orc.propagate(pz, ops, fact, p.c0, 5)
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    # under the field
    c = prop.to_device(p.c0)
    n_steps = 5
    first = 40
    gt = p.g_table(n_steps, first_step=first)
    st = prop.propagate(c, gt)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, n_steps, first_step=first)
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    assert abs(prop.norm(c) - orc.s_norm_sq(ops, p.c0)) <= 1e-9


def test_fixed_iteration_trace_p11(tiny_stress):
    p, prop, ops, fact = tiny_stress
    k = 4
    g = p.g_mid(0)
    x_ref, info = orc.cn_step(ops, fact, p.c0, g, p.dt, p.rtol, p.max_iter, force_iters=k, keep_trace=True)
    c = prop.to_device(p.c0)
    tr = prop.step_forced(c, g, k).cpu().numpy()
    names = ["p", "v", "s", "t", "x", "r", "y", "z"]
    for it in range(k):
        for q, nm in enumerate(names):
            ref = info.trace[it][nm]
            scale = max(np.linalg.norm(ref), 1e-300)
            # residual-like vectors shrink by orders of magnitude per iteration: compare against ||b||-scaled floor
            tol = 1e-11 * max(1.0, np.linalg.norm(info.trace[0]["p"]) / scale) if nm in ("s", "r", "t", "v", "p", "y", "z") else 1e-11
            assert np.linalg.norm(tr[it, q] - ref) / scale <= min(tol, 1e-6), (it, nm)
    assert rel(c.cpu().numpy(), x_ref) <= 1e-11


def test_determinism_p12(smallmed):
    p, prop, _, _ = smallmed
    outs = []
    for _ in range(2):
        c = prop.to_device(p.c0)
        prop.propagate(c, p.g_table(4))
        outs.append(c.cpu().numpy().copy())
    assert np.array_equal(outs[0], outs[1])


def test_speculation_stall_and_resume():
    """A hard system (strong field) needs more iterations than are speculated per step: the stall latch, the
    resume path and the growth of nspec must give the same answer as the oracle."""
    p, prop = make("tiny", phase=np.pi / 2, e0=40.0)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 4)
    assert max(i.half_iters for i in infos) > 6
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(4))
    assert st["steps"] == 4
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    prop.close()


def test_noconv_is_reported():
    p, prop = make("tiny", phase=np.pi / 2, e0=40.0, max_iter=1)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(2), check=False)
    assert st["rc"] == -6 and st["status"] == -6 and st["steps"] == 0
    # the handle stays usable: field-free steps converge at once
    st = prop.propagate(c, np.zeros((2, p.n_terms)))
    assert st["steps"] == 2
    prop.close()


def test_time_reversal_p4(tiny_stress):
    from paper_2512_21697_b200 import Tdde
    p, prop, _, _ = tiny_stress
    back = Tdde(p, dt=-p.dt)
    c = prop.to_device(p.c0)
    g = p.g_mid(2)
    prop.step(c, g)
    back.step(c, g)
    assert rel(c.cpu().numpy(), p.c0) <= 10 * p.rtol
    back.close()


def test_propagate_host_roundtrip(tiny_stress):
    p, prop, ops, fact = tiny_stress
    c = p.c0.copy()
    prop.propagate_host(c, p.g_table(3), 3)
    d = prop.to_device(p.c0)
    prop.propagate(d, p.g_table(3))
    assert np.array_equal(c, d.cpu().numpy())


def test_sampled_rows_at_bench_size_p10():
    """BASELINE configs[3] (Large) in the launch configuration bench.py times: sampled outputs against the
    oracle's direct summation of the definition (the CSR would need 17 GB)."""
    p, prop = make("large", with_c0=False)
    assert prop.apply_path == "banded"
    import torch
    x = rand_vec(p.n, 21)
    xd = prop.to_device(x)
    g = np.linspace(-1.0, 1.0, p.n_terms)
    y = prop.apply(1.0, 0.5j * p.dt, g, xd).cpu().numpy().reshape(p.n_ang, p.n_rad)
    rng = np.random.default_rng(0)
    ns = 400
    chan = np.concatenate([rng.integers(0, p.n_ang, ns), [0, 0, p.n_ang - 1, p.n_ang - 1, 1, 5, p.n_ang - 6]])
    rad = np.concatenate([rng.integers(0, p.n_rad, ns), [0, p.n_rad - 1, 0, p.n_rad - 1, 5, 6, p.n_rad - 7]])
    ref = orc.apply_rows_sampled(p, 1.0, 0.5j * p.dt, g, x, chan, rad)
    got = y[chan, rad]
    scale = np.sqrt(np.mean(np.abs(ref) ** 2))
    assert np.max(np.abs(got - ref)) / scale <= 1e-12
    # properties that hold at any size: M (M^-1 x) = x, and S-norm of a normalised vector
    z = prop.precond(xd)
    back = prop.apply(1.0, 0.5j * p.dt, np.zeros(p.n_terms), z).cpu().numpy()
    assert rel(back, x) <= 1e-12
    del xd, z
    torch.cuda.empty_cache()
    prop.close()


@pytest.mark.parametrize("ng", ["1", "2"])
def test_apply_both_term_split_variants(ng, monkeypatch):
    """The banded apply exists with one warp group and with the terms split over two; the library picks one by T.
    Force each (TDDE_APPLY_NG is read at tdde_create) on a T = 7 and a T = 5 shape, ragged sizes."""
    from paper_2512_21697_b200 import Tdde
    monkeypatch.setenv("TDDE_APPLY_NG", ng)
    for n_ang, n_r, T in [(150, 29, 7), (70, 41, 5)]:
        p = tdde_inputs.make_synthetic(n_ang=n_ang, n_r=n_r, bandwidth=13, n_terms=T, dt=0.01, n_steps=2, rtol=1e-10,
                                       seed=5, name="split", phase=np.pi / 2, e0=2.0)
        prop = Tdde(p)
        assert prop.apply_path == "banded"
        ops, fact = orc.assemble(p), orc.factor_precond(p)
        x = rand_vec(p.n, 2)
        g = np.linspace(-1.0, 1.0, T)
        y = prop.apply(1.0, 0.5j * p.dt, g, prop.to_device(x)).cpu().numpy()
        assert rel(y, orc.apply(ops, 1.0, 0.5j * p.dt, g, x)) <= 1e-12
        c = prop.to_device(p.c0)
        prop.propagate(c, p.g_table(2))
        c_ref, _ = orc.propagate(p, ops, fact, p.c0, 2)
        assert rel(c.cpu().numpy(), c_ref) <= 1e-9
        prop.close()


def test_sampled_rows_and_properties_at_hbm_scale():
    """BASELINE configs[4] (HBM-scale, the workload bench.py times, two-warp-group apply): sampled outputs against the
    oracle's direct summation, M (M^-1 x) = x, and after 3 CN steps S-norm conservation and the solver's residual."""
    import torch
    p, prop = make("hbm", with_c0=False)
    assert prop.apply_path == "banded"
    x = rand_vec(p.n, 33)
    xd = prop.to_device(x)
    g = np.linspace(-1.0, 1.0, p.n_terms)
    y = prop.apply(1.0, 0.5j * p.dt, g, xd).cpu().numpy().reshape(p.n_ang, p.n_rad)
    rng = np.random.default_rng(1)
    ns = 300
    chan = np.concatenate([rng.integers(0, p.n_ang, ns), [0, 0, p.n_ang - 1, p.n_ang - 1, 3, 7, 127, 128, p.n_ang - 8]])
    rad = np.concatenate([rng.integers(0, p.n_rad, ns), [0, p.n_rad - 1, 0, p.n_rad - 1, 5, 6, 443, 444, p.n_rad - 7]])
    ref = orc.apply_rows_sampled(p, 1.0, 0.5j * p.dt, g, x, chan, rad)
    scale = np.sqrt(np.mean(np.abs(ref) ** 2))
    assert np.max(np.abs(y[chan, rad] - ref)) / scale <= 1e-12
    del y
    z = prop.precond(xd)
    back = prop.apply(1.0, 0.5j * p.dt, np.zeros(p.n_terms), z)
    err = float(torch.linalg.vector_norm(back - xd) / torch.linalg.vector_norm(xd))
    assert err <= 1e-12
    del z, back
    n0 = prop.norm(xd)
    st = prop.propagate(xd, p.g_table(3))
    assert st["steps"] == 3 and st["status"] == 0 and st["rel_res"] <= p.rtol
    assert abs(prop.norm(xd) / n0 - 1.0) <= 30 * p.rtol
    del xd
    torch.cuda.empty_cache()
    prop.close()


def test_paper_variant_matches_oracle(smallmed, tiny):
    """NEXT-2 comparator: CSR assembly (one value per non-zero from Eq. 17) + CSR SpMV must give A x = (S + i tau H) x."""
    for p, prop, ops, _ in (smallmed, tiny):
        x = rand_vec(p.n, 4)
        g = np.linspace(0.3, 1.1, p.n_terms)
        y, ta, ts, nnz = prop.paper_variant(g, prop.to_device(x), reps=2)
        y_ref = orc.apply(ops, 1.0, 0.5j * p.dt, g, x)
        assert rel(y.cpu().numpy(), y_ref) <= 1e-12
        # union pattern of the assembled matrix: (coupled channels) x (band) per row, as SURVEY C2 counts it
        A = (ops.S + 0.5j * p.dt * (ops.H0 + sum(ops.K))).tocsr()
        assert nnz >= A.nnz and ta > 0 and ts > 0


def test_eigenstate_phase_closed_form_p3_on_gpu(hyd):
    """P3 on the CUDA path itself (no oracle in the loop): H0 v = E S v  =>  after N field-free CN steps
    c = ((1 - i tau E) / (1 + i tau E))^N v exactly, and every step takes the ||s|| exit at half-iteration 1."""
    import scipy.linalg as sla
    p, prop, _, _ = hyd
    S, H = p.meta["dense"][2]                     # kappa = +2 block (3d3/2-like), a state other than the fixture's 1s
    E, V = sla.eigh(H, S)
    j = int(np.nonzero(E > -p.meta["c"] ** 2)[0][0]) + 1
    a = p.meta["chans"].index((2, 0.5))
    c0 = np.zeros(p.n, dtype=np.complex128)
    c0[a * p.n_rad:(a + 1) * p.n_rad] = V[:, j]
    N = 20
    c = prop.to_device(c0)
    st = prop.propagate(c, np.zeros((N, p.n_terms)))
    tau = 0.5 * p.dt
    phase = ((1 - 1j * tau * E[j]) / (1 + 1j * tau * E[j])) ** N
    assert rel(c.cpu().numpy(), phase * c0) <= 1e-9
    assert st["half_iters"] == N


def test_breakdown_is_reported_for_non_finite_input(tiny):
    p, prop, _, _ = tiny
    bad = p.c0.copy()
    bad[7] = np.nan
    c = prop.to_device(bad)
    st = prop.propagate(c, p.g_table(2), check=False)
    assert st["rc"] == -5 and st["steps"] == 0
    c = prop.to_device(p.c0)                      # the handle recovers on the next call
    st = prop.propagate(c, p.g_table(2))
    assert st["steps"] == 2 and st["status"] == 0


def test_side_stream_and_two_handles(tiny_stress):
    """A handle bound to a non-default torch stream (the step graph is replayed on the caller's stream) and two live
    handles used alternately must reproduce the default-stream result bit for bit."""
    import torch
    from paper_2512_21697_b200 import Tdde
    p, prop, _, _ = tiny_stress
    ref = prop.to_device(p.c0)
    prop.propagate(ref, p.g_table(8))
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        other = Tdde(p, stream=side)
        c = other.to_device(p.c0)
        side.synchronize()
        for k in range(4):                       # alternate with the default-stream handle, 2 steps at a time
            other.propagate(c, p.g_table(2, first_step=2 * k))
            d = prop.to_device(p.c0)
            prop.propagate(d, p.g_table(1))
        side.synchronize()
    assert np.array_equal(c.cpu().numpy(), ref.cpu().numpy())
    other.close()


def test_step_vs_dense_lu_p1_on_gpu(tiny_stress):
    """P1 on the CUDA path without the oracle: the CN step is the exact solution of the dense system
    (S + i tau H) c1 = (S - i tau H) c0 built with numpy.kron from the boundary-format inputs."""
    p, prop, _, _ = tiny_stress
    n_ang, n_rad = p.n_ang, p.n_rad
    S = np.zeros((p.n, p.n), dtype=np.complex128)
    H = np.zeros_like(S)
    for a in range(n_ang):
        k = p.cls_of_chan[a]
        sl = slice(a * n_rad, (a + 1) * n_rad)
        S[sl, sl] = tdde_inputs.band_to_dense(p.S_band[k])
        H[sl, sl] = tdde_inputs.band_to_dense(p.H0_band[k])
    g = p.g_mid(0)
    for L, t in enumerate(p.terms):
        A = np.zeros((n_ang, n_ang), dtype=np.complex128)
        for a in range(n_ang):
            for q in range(t.A_rowptr[a], t.A_rowptr[a + 1]):
                A[a, t.A_col[q]] += t.A_val[q]
        H += g[L] * np.kron(A, tdde_inputs.band_to_dense(t.R_band))
    tau = 0.5 * p.dt
    c1 = np.linalg.solve(S + 1j * tau * H, (S - 1j * tau * H) @ p.c0)
    c = prop.to_device(p.c0)
    prop.step(c, g)
    assert rel(c.cpu().numpy(), c1) <= 1e-10


# ----------------------------------------------------------------------------------------------------------------
# True residual, bandwidth / term-count coverage of the propagation, degenerate exits (VERDICT r1, weak #1 c-e)
def _true_rel_residual(p, prop, c0, c1, g):
    """||b - A c1|| / ||b|| with b = (S - i tau H) c0 and A = S + i tau H, both through tdde_apply (full operator)."""
    import torch
    tau = 0.5 * p.dt
    b = prop.apply(1.0, -1j * tau, g, c0)
    Ax = prop.apply(1.0, +1j * tau, g, c1)
    return float(torch.linalg.vector_norm(b - Ax) / torch.linalg.vector_norm(b))


@pytest.mark.parametrize("kw", [dict(), dict(s_q=0.45), dict(s_q=0.6), dict(h0_scale=300.0), dict(h0_scale=3e4, s_q=0.45)])
def test_true_residual_at_exit(kw):
    """The in-iteration applies of the banded path may use A y = p + i tau (coupling) y (exact up to the rounding of the
    solve M y = p); the residual the solver tests is the recursive one.  Recompute the TRUE residual ||b - A x|| / ||b||
    with the full operator after each step, on well-conditioned, worse-conditioned (S decay 0.45 / 0.6) and stiff
    (tau |H0| >> |S|) field-free blocks, and compare the state with the oracle."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(name="resid", n_ang=70, n_r=90, bandwidth=13, n_terms=5, dt=0.005, n_steps=3,
                                   rtol=1e-10, seed=21, phase=np.pi / 2, e0=2.0, **kw)
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c = prop.to_device(p.c0)
    c_ref = p.c0.copy()
    for s in range(p.n_steps):
        c_prev = c.clone()
        g = p.g_mid(s)
        st = prop.step(c, g)
        assert st["status"] == 0 and st["half_iters"] >= 1
        r_true = _true_rel_residual(p, prop, c_prev, c, g)
        assert r_true <= 1.5 * p.rtol, (kw, s, r_true, st["rel_res"])
        c_ref, info = orc.cn_step(ops, fact, c_ref, g, p.dt, p.rtol, p.max_iter)
    if "h0_scale" not in kw:      # stiff blocks: cond(A) x rtol exceeds 1e-9, two converged solves may differ by more
        assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    prop.close()


@pytest.mark.parametrize("ng", ["1", "2"])
@pytest.mark.parametrize("bw", [7, 19])
def test_propagation_bandwidth_7_and_19_t7(bw, ng, monkeypatch):
    """W = 3 and W = 9 with T = 7 (the shapes of the HBM-scale bandwidth sweep), both term-split variants: full
    propagation against the oracle, not only apply + preconditioner."""
    from paper_2512_21697_b200 import Tdde
    monkeypatch.setenv("TDDE_APPLY_NG", ng)
    p = tdde_inputs.make_synthetic(name="bw", n_ang=150, n_r=45, bandwidth=bw, n_terms=7, dt=0.004, n_steps=4, rtol=1e-10,
                                   seed=31, phase=np.pi / 2, e0=2.0)
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, p.n_steps)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(p.n_steps))
    assert st["steps"] == p.n_steps and st["status"] == 0
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    assert abs(st["half_iters"] - sum(i.half_iters for i in infos)) <= p.n_steps
    prop.close()


def test_zero_iteration_exit_and_zero_state():
    """||r0|| <= rtol ||b|| at the start of a step: no iteration runs and c is returned unchanged (C4, first test); with
    c = 0 both norms vanish (nb2 = 0) and the step must still complete with status ok."""
    p, prop = make("tiny", rtol=0.5)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 2)
    assert [i.half_iters for i in infos] == [0, 0]
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(2))
    assert st["steps"] == 2 and st["half_iters"] == 0 and st["status"] == 0
    assert np.array_equal(c.cpu().numpy(), p.c0) and np.array_equal(c_ref, p.c0)
    prop.close()
    p, prop = make("tiny")
    z = prop.to_device(np.zeros(p.n, dtype=np.complex128))
    st = prop.propagate(z, p.g_table(3))
    assert st["steps"] == 3 and st["status"] == 0 and st["half_iters"] == 0
    assert not np.any(z.cpu().numpy())
    assert prop.norm(z) == 0.0
    prop.close()


@pytest.mark.parametrize("bw", [7, 27])
def test_no_coupling_terms(bw):
    """n_terms = 0 (tdde.h allows it): H = H0, the preconditioner is exact, every step takes the ||s|| exit."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(name="t0", n_ang=37, n_r=40, bandwidth=bw, n_terms=0, dt=0.01, n_steps=3, rtol=1e-11, seed=8)
    prop = Tdde(p)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x = rand_vec(p.n, 3)
    y = prop.apply(0.5, 1.0 - 1.0j, np.zeros(0), prop.to_device(x)).cpu().numpy()
    assert rel(y, orc.apply(ops, 0.5, 1.0 - 1.0j, np.zeros(0), x)) <= 1e-12
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 3)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, np.zeros((3, 0)))
    assert st["steps"] == 3 and st["half_iters"] == 3 == sum(i.half_iters for i in infos)
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    prop.close()


@pytest.mark.parametrize("bw,T", [(9, 3), (11, 4), (15, 6), (5, 2), (7, 6), (13, 1)])
def test_untemplated_bandwidths_and_term_counts(bw, T):
    """Half-bandwidths outside {3, 6, 9, 13} (w = 4, 5, 7, 2) and T = 1, 4, 6: banded couplings that are not one of the instantiated
    shapes FIT inside one (zero-filled slots, padded bands) and stay on the register-resident kernel; apply, preconditioner and
    propagation must match the oracle."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(name="odd", n_ang=75, n_r=33, bandwidth=bw, n_terms=T, dt=0.005, n_steps=3, rtol=1e-10,
                                   seed=bw, phase=np.pi / 2, e0=2.0)
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x = rand_vec(p.n, 6)
    g = np.linspace(0.4, 1.3, T)
    y = prop.apply(1.0, 0.5j * p.dt, g, prop.to_device(x)).cpu().numpy()
    assert rel(y, orc.apply(ops, 1.0, 0.5j * p.dt, g, x)) <= 1e-12
    z = prop.precond(prop.to_device(x)).cpu().numpy()
    assert rel(z, orc.apply_precond(fact, x)) <= 1e-12
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, p.n_steps)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(p.n_steps))
    assert st["steps"] == p.n_steps and rel(c.cpu().numpy(), c_ref) <= 1e-9
    prop.close()


def test_banded_fit_with_permuted_and_thinned_terms():
    """Terms given in an order that is not ascending in reach, with some offsets missing and per-term bandwidths below w0: the
    structure fit re-slots them into an instantiated shape; g is given per caller term and must follow its term."""
    from paper_2512_21697_b200 import Tdde
    base = tdde_inputs.make_synthetic(name="perm", n_ang=140, n_r=31, bandwidth=13, n_terms=5, dt=0.005, n_steps=3, rtol=1e-10, seed=14,
                                      phase=np.pi / 2, e0=2.0)
    rng = np.random.default_rng(3)
    order = [3, 0, 4, 1]                                         # four of the five terms, shuffled (reaches 4, 1, 5, 2)
    terms = []
    for L in order:
        t = base.terms[L]
        keep = np.ones(len(t.A_col), dtype=bool)
        rows = np.repeat(np.arange(base.n_ang), np.diff(t.A_rowptr))
        keep &= ~((np.abs(t.A_col - rows) == 2) & (L == 3))      # drop the offsets +-2 of the reach-4 term (stays Hermitian)
        rowptr = np.concatenate([[0], np.cumsum(np.bincount(rows[keep], minlength=base.n_ang))]).astype(np.int32)
        w = 6 if L != 0 else 4                                   # one term with a narrower radial band
        R = t.R_band if w == 6 else np.ascontiguousarray(t.R_band[:, 2:-2])
        terms.append(tdde_inputs.Term(w=w, R_band=R, A_rowptr=rowptr, A_col=t.A_col[keep], A_val=t.A_val[keep]))
    amps = np.array([0.7, -1.3, 0.4, 2.1])
    d = dict(base.__dict__)
    d.update(terms=terms, g_of_t=lambda t, _a=amps: _a * np.cos(0.057 * t))
    p = tdde_inputs.Problem(**d)
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x = rand_vec(p.n, 6)
    for g in (amps, np.array([1.0, 0.0, 0.0, 0.0]), np.array([0.0, 0.0, 1.0, 0.0])):
        y = prop.apply(1.0, 0.5j * p.dt, g, prop.to_device(x)).cpu().numpy()
        assert rel(y, orc.apply(ops, 1.0, 0.5j * p.dt, g, x)) <= 1e-12, g
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 3)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(3))
    assert st["steps"] == 3 and rel(c.cpu().numpy(), c_ref) <= 1e-9
    tr = prop.step_forced(prop.to_device(p.c0), p.g_mid(0), 1, trace=False)
    prop.close()


# ----------------------------------------------------------------------------------------------------------------
# The three apply kernels: banded (register A_L), staged (sparse A_L in shared memory), generic (unstaged fall-back)
def _random_sparse_problem(seed, n_ang, n_r, bandwidths, nnz_row, w0=None, dup=False):
    """Hermitian-sum coupling with arbitrary sparse (non-banded) A_L, per-term bandwidths, optional duplicate CSR entries."""
    rng = np.random.default_rng(seed)
    base = tdde_inputs.make_synthetic(name="sp", n_ang=n_ang, n_r=n_r, bandwidth=2 * (w0 or max(bandwidths)) + 1, n_terms=0, dt=0.004,
                                      n_steps=3, rtol=1e-10, seed=seed)
    terms = []
    for w in bandwidths:
        dense = np.zeros((n_ang, n_ang), dtype=np.complex128)
        for a in range(n_ang):
            cols = rng.choice(n_ang, size=min(nnz_row, n_ang), replace=False)
            dense[a, cols] += rng.standard_normal(len(cols)) + 1j * rng.standard_normal(len(cols))
        dense = 0.5 * (dense + dense.conj().T)                      # each term Hermitian (its R_L is, too)
        rowptr, col, val = [0], [], []
        for a in range(n_ang):
            nz = np.nonzero(dense[a])[0]
            for cc in nz:
                if dup and rng.random() < 0.3:                        # split one entry into two CSR entries of the same column
                    col += [cc, cc]; val += [0.25 * dense[a, cc], 0.75 * dense[a, cc]]
                else:
                    col.append(cc); val.append(dense[a, cc])
            rowptr.append(len(col))
        R = tdde_inputs.synthetic.herm_band(rng, base.n_rad, w)
        terms.append(tdde_inputs.Term(w=w, R_band=R, A_rowptr=np.asarray(rowptr, np.int32), A_col=np.asarray(col, np.int32),
                                      A_val=np.asarray(val, np.complex128)))
    T = len(terms)
    d = dict(base.__dict__)
    d.update(terms=terms, g_of_t=lambda t, _T=T: np.full(_T, 0.3 * np.cos(0.057 * t)))
    return tdde_inputs.Problem(**d)


@pytest.mark.parametrize("case", [dict(n_ang=50, n_r=30, bandwidths=[2, 4, 6], nnz_row=3, dup=True),          # per-term widths, duplicates
                                  dict(n_ang=300, n_r=25, bandwidths=[6, 6, 6], nnz_row=2),                   # wide reach: whole-row x tile
                                  dict(n_ang=37, n_r=40, bandwidths=[13] * 8, nnz_row=1),                     # hydrogen-like: w = 13, T = 8
                                  dict(n_ang=200, n_r=20, bandwidths=[3], nnz_row=1, w0=9)])                  # block band wider than the term's
def test_staged_sparse_apply_path(case):
    from paper_2512_21697_b200 import Tdde
    p = _random_sparse_problem(41, **case)
    prop = Tdde(p)
    assert prop.apply_path == "staged"
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x = rand_vec(p.n, 8)
    g = np.linspace(0.4, 1.2, p.n_terms)
    for alpha, beta in [(1.0, 0.5j * p.dt), (0.3 - 0.2j, 1.0 + 0.5j)]:
        y = prop.apply(alpha, beta, g, prop.to_device(x)).cpu().numpy()
        assert rel(y, orc.apply(ops, alpha, beta, g, x)) <= 1e-12, case
    assert abs(prop.norm(prop.to_device(x)) - orc.s_norm_sq(ops, x)) <= 1e-12 * orc.s_norm_sq(ops, x)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 3)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(3))
    assert st["steps"] == 3 and rel(c.cpu().numpy(), c_ref) <= 1e-9
    prop.close()


def test_generic_fallback_path_and_bounded_grid(monkeypatch):
    """The unstaged generic kernel (forced here; otherwise only reached for w > 13 or couplings too dense for shared memory):
    parity, and a shape with more (row, channel-block) work items than reduction slots (70400 > 65536)."""
    from paper_2512_21697_b200 import Tdde
    monkeypatch.setenv("TDDE_NO_STAGED", "1")
    monkeypatch.setenv("TDDE_APPLY_PATH", "0")
    p = _random_sparse_problem(43, n_ang=60, n_r=25, bandwidths=[4, 6], nnz_row=3)
    prop = Tdde(p)
    assert prop.apply_path == "generic"
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x = rand_vec(p.n, 2)
    g = np.array([0.7, -0.4])
    y = prop.apply(1.0, 0.5j * p.dt, g, prop.to_device(x)).cpu().numpy()
    assert rel(y, orc.apply(ops, 1.0, 0.5j * p.dt, g, x)) <= 1e-12
    c_ref, _ = orc.propagate(p, ops, fact, p.c0, 3)
    c = prop.to_device(p.c0)
    prop.propagate(c, p.g_table(3))
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    prop.close()
    # 16 channel blocks x 4400 rows = 70400 work items; w = 4 is not a banded-kernel width
    big = tdde_inputs.make_synthetic(name="biggrid", n_ang=2000, n_r=2200, bandwidth=9, n_terms=1, dt=0.002, n_steps=1, rtol=1e-10, seed=5,
                                     with_c0=False)
    prop = Tdde(big)
    assert prop.apply_path == "generic"
    x = rand_vec(big.n, 4)
    xd = prop.to_device(x)
    n_gpu = prop.norm(xd)                                              # S-only apply with the fused grid reduction
    X = x.reshape(big.n_ang, big.n_rad)
    ref = 0.0
    w = big.w0
    for d in range(-w, w + 1):
        lo, hi = max(0, -d), min(big.n_rad, big.n_rad - d)
        ref += float(np.real(np.sum(np.conj(X[:, lo:hi]) * (0.3 ** abs(d)) * X[:, lo + d:hi + d])))
    assert abs(n_gpu - ref) <= 1e-11 * ref
    g = np.array([0.9])
    y = prop.apply(1.0, 0.5j * big.dt, g, xd).cpu().numpy().reshape(big.n_ang, big.n_rad)
    rng = np.random.default_rng(0)
    chan, rad = rng.integers(0, big.n_ang, 200), rng.integers(0, big.n_rad, 200)
    refs = orc.apply_rows_sampled(big, 1.0, 0.5j * big.dt, g, x, chan, rad)
    assert np.max(np.abs(y[chan, rad] - refs)) <= 1e-12 * np.sqrt(np.mean(np.abs(refs) ** 2))
    prop.close()


# ----------------------------------------------------------------------------------------------------------------
# NEXT-1: the paper-shaped non-dipole operator set (x-polarised, mu' = mu +- 1, l <= l_max, 8 Kronecker terms per l)
def test_nondipole_operator_set_parity():
    """Eq. 17-18 of the paper (H^theta_l from Clebsch-Gordan x 3j, 24 Kronecker terms for l_max = 2, real Dirac DKB blocks,
    seeded stand-ins for the radial g^n_l): apply <= 1e-12 and propagation <= 1e-9 against the oracle, on the staged sparse-A kernel."""
    from paper_2512_21697_b200 import Tdde
    from tdde_inputs import nondipole as nd
    p = nd.set_ground_state(nd.make_nondipole(kappa_max=6, l_max=2, n_r=30))
    prop = Tdde(p)
    assert prop.apply_path == "staged" and p.n_terms == 24
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    x = rand_vec(p.n, 12)
    xd = prop.to_device(x)
    for alpha, beta, g in [(1.0, 0.5j * p.dt, p.g_mid(70)), (0.2 + 0.1j, 1.0 - 0.5j, np.linspace(-1.0, 1.0, p.n_terms))]:
        y = prop.apply(alpha, beta, g, xd).cpu().numpy()
        assert rel(y, orc.apply(ops, alpha, beta, np.asarray(g, float), x)) <= 1e-12
    z = prop.precond(xd).cpu().numpy()
    assert rel(z, orc.apply_precond(fact, x)) <= 1e-12
    n_steps, first = 4, 60
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, n_steps, first_step=first)
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(n_steps, first_step=first))
    assert st["steps"] == n_steps and st["status"] == 0
    assert rel(c.cpu().numpy(), c_ref) <= 1e-9
    assert abs(st["half_iters"] - sum(i.half_iters for i in infos)) <= n_steps
    assert abs(prop.norm(c) - orc.s_norm_sq(ops, p.c0)) <= 1e-9
    prop.close()


def test_nondipole_kappa15_sampled_rows():
    """kappa_max = 15 (480 channels, 24 terms, up to 11 couplings per row and term): outputs sampled against the oracle's
    direct summation of the definition; S-norm conservation over a few steps under the field."""
    from paper_2512_21697_b200 import Tdde
    from tdde_inputs import nondipole as nd
    p = nd.set_ground_state(nd.make_nondipole(kappa_max=15, l_max=2, n_r=40))
    prop = Tdde(p)
    assert prop.apply_path == "staged" and p.n_ang == 480
    x = rand_vec(p.n, 13)
    g = np.linspace(0.3, 1.1, p.n_terms)
    y = prop.apply(1.0, 0.5j * p.dt, g, prop.to_device(x)).cpu().numpy().reshape(p.n_ang, p.n_rad)
    rng = np.random.default_rng(2)
    chan = np.concatenate([rng.integers(0, p.n_ang, 150), [0, 1, p.n_ang - 1, 127, 128, 255, 256]])
    rad = np.concatenate([rng.integers(0, p.n_rad, 150), [0, p.n_rad - 1, 5, 13, 14, 40, 41]])
    ref = orc.apply_rows_sampled(p, 1.0, 0.5j * p.dt, g, x, chan, rad)
    assert np.max(np.abs(y[chan, rad] - ref)) <= 1e-12 * np.sqrt(np.mean(np.abs(ref) ** 2))
    c = prop.to_device(p.c0)
    n0 = prop.norm(c)
    st = prop.propagate(c, p.g_table(3, first_step=60))
    assert st["steps"] == 3 and st["status"] == 0 and st["half_iters"] >= 6
    assert abs(prop.norm(c) - n0) <= 1e-9
    prop.close()


def test_projection_on_eigenstates_next4(hyd):
    """tdde_project (Eq. 33): |<psi_{kappa,e}| S |c_a>|^2 for every channel and eigenstate, against the
    oracle; on the hydrogen basis the propagated 1s state keeps its weight on the 1s eigenstate when the field is off."""
    import scipy.linalg as sla
    p, prop, ops, fact = hyd
    V = np.zeros((p.n_cls, p.n_rad, p.n_rad), dtype=np.complex128)
    for k, kap in enumerate(p.meta["kappas"]):
        S, H = p.meta["dense"][kap]
        _, vec = sla.eigh(H, S)
        V[k] = vec.T
    prop.set_eigenstates(V)
    x = rand_vec(p.n, 17)
    P = prop.project(prop.to_device(x))
    ref = orc.project(p, V, x)
    assert np.max(np.abs(P - ref)) <= 1e-12 * np.max(ref)
    c = prop.to_device(p.c0)
    prop.propagate(c, np.zeros((10, p.n_terms)))
    P = prop.project(c)
    a = p.meta["chans"].index((-1, 0.5))
    S1, H1 = p.meta["dense"][-1]
    E1 = sla.eigh(H1, S1, eigvals_only=True)
    j = int(np.nonzero(E1 > -p.meta["c"] ** 2)[0][0])
    assert abs(P[a, j] - 1.0) <= 1e-9 and abs(P.sum() - 1.0) <= 1e-9
    # fewer states than basis functions
    prop.set_eigenstates(V[:, 5:45, :])
    P2 = prop.project(prop.to_device(x))
    assert np.max(np.abs(P2 - ref[:, 5:45])) <= 1e-12 * np.max(ref)


def test_device_eigensolve_next4(hyd):
    """tdde_eigensolve (Eq. 19-20): all eigenpairs of the eight hydrogen pencils (H0_k, S_k), n_rad = 400,
    against LAPACK through the oracle, the Sommerfeld closed form for the bound levels, the pencil residual and S-orthonormality;
    the device's own eigenvectors then feed tdde_project."""
    from paper_2512_21697_b200 import eigensolve
    p, prop, ops, fact = hyd
    E_ref, V_ref = orc.eigenstates(p)
    E, V = eigensolve(p.S_band, p.H0_band)
    scale = np.max(np.abs(E_ref))                              # ~ 2 c^2 + the stiffest pseudo-continuum state
    assert np.max(np.abs(E - E_ref)) <= 1e-12 * scale
    c2 = p.meta["c"] ** 2
    k1 = p.meta["kappas"].index(-1)
    e1s = E[k1][E[k1] > -c2][0]
    assert abs(e1s - c2 * (np.sqrt(1.0 - 1.0 / c2) - 1.0)) <= 1e-9          # Dirac 1s1/2: c^2 (sqrt(1 - (Z/c)^2) - 1)
    for k in range(p.n_cls):
        S, H = tdde_inputs.band_to_dense(p.S_band[k]), tdde_inputs.band_to_dense(p.H0_band[k])
        R = H @ V[k].T - (S @ V[k].T) * E[k][None, :]
        assert np.linalg.norm(R) <= 1e-11 * np.linalg.norm(H) * np.sqrt(p.n_rad)
        assert np.max(np.abs(V[k].conj() @ S @ V[k].T - np.eye(p.n_rad))) <= 1e-9
    # projections with the device's eigenvectors: the same probabilities as with LAPACK's up to the conditioning of individual
    # eigenvectors (eps |H| / gap: the spectrum spans 2 c^2 with gaps far below 1), and the same total per channel to rounding
    prop.set_eigenstates(V)
    x = rand_vec(p.n, 23)
    P = prop.project(prop.to_device(x))
    P_ref = orc.project(p, V_ref, x)
    assert np.max(np.abs(P - P_ref)) <= 1e-6 * np.max(P)
    assert np.max(np.abs(P.sum(axis=1) - P_ref.sum(axis=1))) <= 1e-10 * np.max(P_ref.sum(axis=1))
    # a complex Hermitian pencil with a ragged size (odd n: one bye per Jacobi round)
    q = tdde_inputs.make_synthetic(name="eig", n_ang=5, n_r=23, bandwidth=7, n_terms=0, dt=0.01, n_steps=1, rtol=1e-10, seed=9, with_c0=False)
    q.S_band = q.S_band[:, :45].copy(); q.H0_band = q.H0_band[:, :45].copy()
    for band in (q.S_band, q.H0_band):                        # entries pointing outside the truncated matrix are ignored by contract
        w = q.w0
        for i in range(45):
            for d in range(-w, w + 1):
                if i + d < 0 or i + d >= 45:
                    band[:, i, d + w] = 0.0
    q.n_rad = 45
    Eq_ref, _ = orc.eigenstates(q)
    Eq, Vq = eigensolve(q.S_band, q.H0_band)
    assert np.max(np.abs(Eq - Eq_ref)) <= 1e-12 * np.max(np.abs(Eq_ref))
    S, H = tdde_inputs.band_to_dense(q.S_band[2]), tdde_inputs.band_to_dense(q.H0_band[2])
    assert np.linalg.norm(H @ Vq[2].T - (S @ Vq[2].T) * Eq[2][None, :]) <= 1e-12 * np.linalg.norm(H) * 45


# ---- in-iteration apply (R21 / 4.1): y = addv + beta sum_L g_L (A_L (x) R_L) x, DMMA variant and register-window variant ----
@pytest.mark.parametrize("n_ang,n_r,T,bw,seg", [(257, 53, 7, 13, 0), (100, 41, 7, 19, 16), (130, 37, 5, 13, 8), (96, 64, 7, 13, 24),
                                                (33, 9, 7, 13, 0)])
def test_coupling_apply_parity_mma_and_window(n_ang, n_r, T, bw, seg, monkeypatch):
    """All outputs and the fused sums of the kernel an iteration uses for v = A y, against the oracle's coupling part
    (apply with g minus apply with g = 0), for the DMMA kernel (which=0) and the register-window kernel (which=1): channel counts
    that are not multiples of 8 / 96, radial sizes that are not multiples of 8, several radial segments (TDDE_MMA_SEG)."""
    from paper_2512_21697_b200 import Tdde
    if seg:
        monkeypatch.setenv("TDDE_MMA_SEG", str(seg))
    p = tdde_inputs.make_synthetic(n_ang=n_ang, n_r=n_r, bandwidth=bw, n_terms=T, dt=0.01, n_steps=1, rtol=1e-10, seed=n_ang + T,
                                   name="coupling")
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    ops = orc.assemble(p)
    x, addv, aux = rand_vec(p.n, 11), rand_vec(p.n, 12), rand_vec(p.n, 13)
    g = np.linspace(0.4, 1.7, T)
    beta = 0.3 - 0.8j
    y_ref = addv + orc.apply(ops, 0.0, beta, g, x) - orc.apply(ops, 0.0, beta, np.zeros(T), x)
    for which in (0, 1):
        y, dot, nrm2 = prop.apply_coupling(beta, g, prop.to_device(x), prop.to_device(addv), prop.to_device(aux), which=which)
        y = y.cpu().numpy()
        assert rel(y, y_ref) <= 1e-12, (which, n_ang, n_r, T, bw)
        assert np.max(np.abs(y - y_ref)) <= 1e-12 * np.sqrt(np.mean(np.abs(y_ref) ** 2)) * 50, which
        assert abs(dot - np.vdot(aux, y_ref)) <= 1e-12 * np.linalg.norm(aux) * np.linalg.norm(y_ref), which
        assert abs(nrm2 - np.vdot(y_ref, y_ref).real) <= 1e-12 * np.vdot(y_ref, y_ref).real, which
    prop.close()


def test_mma_and_window_propagation_agree(monkeypatch):
    """Same propagation with the DMMA kernel and with TDDE_NO_MMA=1: same iteration counts, states equal to rounding, both within
    1e-9 of the oracle."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(n_ang=200, n_r=45, bandwidth=13, n_terms=7, dt=0.01, n_steps=4, rtol=1e-10, seed=77, name="mma_prop",
                                   phase=np.pi / 2, e0=2.0)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 4)
    out = []
    for no_mma in (False, True):
        if no_mma:
            monkeypatch.setenv("TDDE_NO_MMA", "1")
        prop = Tdde(p)
        c = prop.to_device(p.c0)
        st = prop.propagate(c, p.g_table(4))
        out.append((c.cpu().numpy(), st["half_iters"]))
        prop.close()
    assert out[0][1] == out[1][1]
    assert rel(out[0][0], out[1][0]) <= 1e-13
    assert rel(out[0][0], c_ref) <= 1e-9 and rel(out[1][0], c_ref) <= 1e-9
    assert abs(out[0][1] - sum(i.half_iters for i in infos)) <= 4


@pytest.mark.parametrize("bw,T", [(13, 7), (19, 7), (13, 5), (7, 7)])
def test_split_start_of_step_matches_single_apply_start(bw, T, monkeypatch):
    """Start of a step as block pass (r = -i dt H0 c, s = S c) + DMMA coupling apply with the ||b||^2 / ||r0||^2 epilogue
    (TDDE_SPLIT_START forces it for every shape that has a DMMA kernel) against the single H-apply + S-apply start: same iteration
    counts, states equal to rounding, both within 1e-9 of the oracle; radial size not a multiple of 8, ragged channel count."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(n_ang=230, n_r=43, bandwidth=bw, n_terms=T, dt=0.01, n_steps=3, rtol=1e-10, seed=5 + bw, name="split",
                                   phase=np.pi / 2, e0=1.5)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, 3)
    out = []
    for env in ("TDDE_SPLIT_START", "TDDE_NO_SPLIT_START"):
        monkeypatch.delenv("TDDE_SPLIT_START", raising=False)
        monkeypatch.setenv(env, "1")
        prop = Tdde(p)
        c = prop.to_device(p.c0)
        st = prop.propagate(c, p.g_table(3))
        out.append((c.cpu().numpy(), st["half_iters"], st["rel_res"]))
        prop.close()
    assert out[0][1] == out[1][1]
    assert rel(out[0][0], out[1][0]) <= 1e-13
    assert rel(out[0][0], c_ref) <= 1e-9 and rel(out[1][0], c_ref) <= 1e-9
