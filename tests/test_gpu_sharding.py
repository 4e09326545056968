"""NEXT-3 device path (include/tdde.h tdde_group_*): channel-slab shards driven in lock step.
One GPU: every shard of the job lives in this process on one stream (device copies stand in for the NVLink transfers, a summing kernel
for the all-reduce), which exercises the ownership masks, the halo exchange, the split reductions and the lock-step driver; the NCCL
path is exercised with a world of one (library loading, communicator, all-reduce, finalisation)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import tdde_inputs  # noqa: E402
from oracle import tdde_oracle as orc  # noqa: E402

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _run_sharded(p, world, n_steps, nccl=False):
    from paper_2512_21697_b200 import Tdde, TddeGroup, nccl_unique_id, sharding
    parts = sharding.shard_specs(p, world)
    shards = [Tdde(pl) for _, pl, _ in parts]
    grp = TddeGroup(shards, [sp for _, _, sp in parts], nccl_unique_id() if nccl else None)
    c0 = p.c0.reshape(p.n_ang, p.n_rad)
    cs = []
    for (plan, _, _), sh in zip(parts, shards):
        loc = c0[plan.halo_lo:plan.halo_hi].copy()
        loc[:plan.lo - plan.halo_lo] = 77.0            # halo entries of the caller's vector are ignored: poison them
        loc[plan.hi - plan.halo_lo:] = -55.0
        cs.append(sh.to_device(loc.reshape(-1)))
    st = grp.propagate(cs, p.g_table(n_steps))
    out = np.zeros((p.n_ang, p.n_rad), dtype=np.complex128)
    for (plan, _, _), c in zip(parts, cs):
        out[plan.lo:plan.hi] = c.cpu().numpy().reshape(plan.n_local, p.n_rad)[plan.own_slice]
    grp.close()
    for sh in shards:
        sh.close()
    return out.reshape(-1), st


@pytest.mark.parametrize("n_ang,T,bw,world,gather", [(70, 3, 7, 2, True), (150, 7, 13, 3, True), (150, 7, 13, 3, False), (97, 5, 13, 2, True),
                                                     (64, 7, 19, 4, True), (64, 7, 19, 4, False)])
def test_sharded_propagation_matches_unsharded_oracle(n_ang, T, bw, world, gather, monkeypatch):
    """gather: the in-iteration applies of shards that run k_apply_mma fetch their halo columns straight from the neighbours' vectors
    (k_apply_mma<GATHER>); TDDE_NO_GATHER=1 keeps the separate halo copies for the same problems; T = 3 has no DMMA kernel (copies)."""
    if not gather:
        monkeypatch.setenv("TDDE_NO_GATHER", "1")
    n_steps = 3
    p = tdde_inputs.make_synthetic(n_ang=n_ang, n_r=21, bandwidth=bw, n_terms=T, dt=0.01, n_steps=n_steps, rtol=1e-10, seed=n_ang,
                                   tiny_offsets=(T == 3), name="shard", phase=np.pi / 2, e0=1.5)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, n_steps)
    c, st = _run_sharded(p, world, n_steps)
    assert st["steps"] == n_steps and st["status"] == 0
    assert rel(c, c_ref) <= 1e-9
    assert abs(st["half_iters"] - sum(i.half_iters for i in infos)) <= n_steps
    # and against the unsharded CUDA path: same algorithm, only the summation order of the inner products differs
    from paper_2512_21697_b200 import Tdde
    prop = Tdde(p)
    cd = prop.to_device(p.c0)
    st1 = prop.propagate(cd, p.g_table(n_steps))
    assert rel(c, cd.cpu().numpy()) <= 1e-10
    assert abs(st["half_iters"] - st1["half_iters"]) <= n_steps
    prop.close()


def test_sharded_hydrogen_staged_path():
    """General sparse couplings (staged kernel) in two shards: the z-dipole hydrogen problem, 2 steps at the field maximum."""
    p = tdde_inputs.make_hydrogen(n_r=40, r_max=40.0, kappa_max=3, e0=0.5, t_offset=55.0)
    rng = np.random.default_rng(1)
    p.c0[:] = rng.standard_normal(p.n) + 1j * rng.standard_normal(p.n)
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, _ = orc.propagate(p, ops, fact, p.c0, 2)
    c, st = _run_sharded(p, 2, 2)
    assert st["status"] == 0 and rel(c, c_ref) <= 1e-9


def test_group_over_nccl_world_of_one():
    """One shard that owns everything, communicator from a fresh NCCL id: the all-reduce and the deferred scalar update run through
    libnccl; the result must equal the plain single-GPU propagation to rounding (same kernels, same summation order)."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(n_ang=60, n_r=20, bandwidth=13, n_terms=5, dt=0.01, n_steps=3, rtol=1e-10, seed=3, name="nccl1",
                                   phase=np.pi / 2, e0=1.0)
    c, st = _run_sharded(p, 1, 3, nccl=True)
    prop = Tdde(p)
    cd = prop.to_device(p.c0)
    st1 = prop.propagate(cd, p.g_table(3))
    assert st["half_iters"] == st1["half_iters"]
    assert rel(c, cd.cpu().numpy()) <= 1e-13
    prop.close()


def test_sharded_large_shapes_use_the_dmma_apply_and_fused_updates():
    """2.2 M elements in two shards: the shards run k_apply_mma and the fused update + spike-product kernels (sizes below that use the
    other kernels).  Compared with the unsharded CUDA path (itself held to the oracle in test_gpu_parity_scale.py) and, on sampled output
    rows of the first step's operator, with the oracle's definition."""
    from paper_2512_21697_b200 import Tdde
    p = tdde_inputs.make_synthetic(n_ang=1200, n_r=900, bandwidth=13, n_terms=7, dt=0.005, n_steps=2, rtol=1e-10, seed=9, name="shard_big",
                                   phase=np.pi / 2, e0=1.0)
    c, st = _run_sharded(p, 2, 2)
    prop = Tdde(p)
    assert prop.iter_apply_kernel == "k_apply_mma"
    cd = prop.to_device(p.c0)
    st1 = prop.propagate(cd, p.g_table(2))
    assert st["status"] == 0 and abs(st["half_iters"] - st1["half_iters"]) <= 2
    assert rel(c, cd.cpu().numpy()) <= 1e-10
    assert abs(prop.norm(prop.to_device(c)) - 1.0) <= 1e-9
    prop.close()
