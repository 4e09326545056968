"""GPU parity at the sizes bench.py times: the BASELINE configs themselves against the oracle (not against the
GPU path's own invariants).  Medium runs its full 100 steps against the CSR oracle; Large and HBM-scale, whose CSR
(17 GB / 125 GB) cannot be held, run against the oracle's panel-streamed matrix-free form (oracle.apply_panels /
cn_step_panels, pinned on small problems against numpy.kron in tests/test_oracle_pins.py).

Tolerances are north_star's: relative L2 <= 1e-12 per operator apply, <= 1e-9 on the wavefunction after the propagation.
"""
import numpy as np
import pytest

import tdde_inputs
from oracle import tdde_oracle as orc

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def rand_vec(n, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal(2 * n).view(np.complex128).copy()


def test_medium_full_100_steps_vs_csr_oracle():
    """BASELINE configs[2] exactly (512 x 1000, w = 6, T = 5, dt 0.005, rtol 1e-10, seed 1), all 100 CN steps, against the
    oracle's textbook BiCGSTAB on the explicitly assembled CSR operators (S, H0 and the five K_L; 0.2 G non-zeros)."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_config("medium")
    assert (p.n_ang, p.n_rad, p.w0, p.n_terms, p.n_steps, p.rtol) == (512, 1000, 6, 5, 100, 1e-10)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, p.n_steps, assembled=False)
    assert all(i.status == "ok" for i in infos)
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(p.n_steps))
    assert st["steps"] == p.n_steps and st["status"] == 0
    err = rel(c.cpu().numpy(), c_ref)
    assert err <= 1e-9, err
    assert abs(st["half_iters"] - sum(i.half_iters for i in infos)) <= p.n_steps
    assert abs(prop.norm(c) - orc.s_norm_sq(ops, c_ref)) <= 1e-9
    prop.close()


def test_large_first_steps_vs_matrix_free_oracle():
    """BASELINE configs[3] (3000 x 2000, T = 5): the first 6 of its 50 steps against the oracle's matrix-free form (the
    CSR of the K_L would need ~25 GB plus as much again while it is built; 6 steps keep the CPU side near two minutes)."""
    import torch
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_config("large")
    fact = orc.factor_precond(p)
    n_steps = 6
    c_ref = p.c0.copy()
    halves = 0
    for s in range(n_steps):
        c_ref, info = orc.cn_step_panels(p, fact, c_ref, p.g_mid(s), p.dt, p.rtol, p.max_iter)
        assert info.status == "ok"
        halves += info.half_iters
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(n_steps))
    assert st["steps"] == n_steps and st["status"] == 0
    err = rel(c.cpu().numpy(), c_ref)
    assert err <= 1e-9, err
    assert abs(st["half_iters"] - halves) <= n_steps
    del c
    torch.cuda.empty_cache()
    prop.close()


def test_hbm_scale_full_vector_apply_and_steps_vs_oracle():
    """BASELINE configs[4], the workload and launch configuration bench.py times (8000 x 4000, T = 7, two-warp-group
    apply): (i) ONE FULL-VECTOR apply with non-zero g compared over all 3.2e7 outputs with the oracle's panel-streamed
    evaluation of the definition (every CTA seam, radial segment boundary and halo channel included);
    (ii) the first 2 CN steps against the oracle's matrix-free BiCGSTAB."""
    import torch
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_config("hbm")
    prop = Tdde(p)
    assert prop.apply_path == "banded"
    x = rand_vec(p.n, 33)
    g = np.linspace(-1.0, 1.0, p.n_terms)
    xd = prop.to_device(x)
    y = prop.apply(1.0, 0.5j * p.dt, g, xd).cpu().numpy()
    del xd
    y_ref = orc.apply_panels(p, 1.0, 0.5j * p.dt, g, x)
    assert rel(y, y_ref) <= 1e-12
    # element-wise as well: no single output off by more than 1e-12 of the rms output
    assert float(np.max(np.abs(y - y_ref))) <= 1e-12 * float(np.sqrt(np.mean(np.abs(y_ref) ** 2)))
    del y, y_ref, x
    fact = orc.factor_precond(p)
    n_steps = 2
    c_ref = p.c0.copy()
    for s in range(n_steps):
        c_ref, info = orc.cn_step_panels(p, fact, c_ref, p.g_mid(s), p.dt, p.rtol, p.max_iter)
        assert info.status == "ok"
    c = prop.to_device(p.c0)
    st = prop.propagate(c, p.g_table(n_steps))
    assert st["steps"] == n_steps and st["status"] == 0
    err = rel(c.cpu().numpy(), c_ref)
    assert err <= 1e-9, err
    del c
    torch.cuda.empty_cache()
    prop.close()
