"""NEXT-3 host logic: the channel-slab plan of paper_2512_21697_b200/sharding.py
exercised with TWO gloo ranks on CPU.  Each rank holds [halo | owned | halo] channels, gathers the halo slabs of the input vector
before every operator apply, keeps the preconditioner local and all-reduces every inner product over OWNED channels only -- the
protocol the device path would follow -- with the oracle's operator on the rank-local problem standing in for the per-rank
CUDA handle.  The gathered result must equal the unsharded oracle CN step."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _make_problem():
    import tdde_inputs
    return tdde_inputs.make_synthetic(name="shard", n_ang=23, n_r=12, bandwidth=7, n_terms=3, dt=0.01, n_steps=2, rtol=1e-12, seed=5,
                                      phase=np.pi / 2, e0=3.0)


def _allreduce(x):
    t = torch.tensor(np.atleast_1d(np.asarray(x)).view(np.float64).copy())
    dist.all_reduce(t)
    return t.numpy().view(np.asarray(x).dtype)


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    from oracle import tdde_oracle as orc
    from paper_2512_21697_b200 import sharding
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = _make_problem()
    plans = sharding.plan_slabs(p, world)
    plan = plans[rank]
    bounds = sharding.slab_bounds(p.n_ang, world)
    pl = sharding.local_problem(p, plan)
    ops = orc.assemble(pl)
    fact = orc.factor_precond(pl)
    n_rad, own = p.n_rad, plan.own_slice
    max_slab = max(bounds[r + 1] - bounds[r] for r in range(world))

    def exchange(x_loc):
        """Refresh the halo channels of a local vector from their owners (all-gather of the owned slabs, as on NVSwitch)."""
        X = x_loc.reshape(plan.n_local, n_rad)
        mine = np.zeros((max_slab, n_rad), dtype=np.complex128)
        mine[:plan.hi - plan.lo] = X[own]
        bufs = [torch.zeros(max_slab, n_rad, dtype=torch.complex128) for _ in range(world)]
        dist.all_gather(bufs, torch.from_numpy(mine))
        for r, a, b in plan.needs_from(bounds):
            X[a - plan.halo_lo:b - plan.halo_lo] = bufs[r].numpy()[a - bounds[r]:b - bounds[r]]
        return X.reshape(-1)

    def owned(x_loc):
        return x_loc.reshape(plan.n_local, n_rad)[own].reshape(-1)

    def vdot(u, v):      # inner product over owned channels, summed over the ranks
        return _allreduce(np.array([np.vdot(owned(u), owned(v))]))[0]

    def A_mul(g, tau, x_loc, sign=+1):
        y = orc.apply(ops, 1.0, sign * 1j * tau, g, exchange(x_loc.copy()))
        Y = y.reshape(plan.n_local, n_rad)
        mask = np.zeros(plan.n_local, dtype=bool)
        mask[own] = True
        Y[~mask] = 0.0                       # halo rows are another rank's outputs
        return Y.reshape(-1)

    c = pl.c0.copy()
    for step in range(p.n_steps):
        g, tau = p.g_mid(step), 0.5 * p.dt
        b = A_mul(g, tau, c, -1)
        # the oracle's BiCGSTAB with rank-global inner products (same order of operations, C4)
        x = c.copy()
        r = b - A_mul(g, tau, x)
        rhat = r.copy()
        nb = np.sqrt(vdot(b, b).real)
        rho_old = alpha = omega = 1.0 + 0.0j
        v = np.zeros_like(x); pp = np.zeros_like(x)
        for _ in range(p.max_iter):
            rho = vdot(rhat, r)
            beta = (rho / rho_old) * (alpha / omega)
            rho_old = rho
            pp = r + beta * (pp - omega * v)
            y = orc.apply_precond(fact, pp)                 # block-diagonal over channels: rank-local
            v = A_mul(g, tau, y)
            alpha = rho / vdot(rhat, v)
            s = r - alpha * v
            if np.sqrt(vdot(s, s).real) <= p.rtol * nb:
                x = x + alpha * y
                break
            z = orc.apply_precond(fact, s)
            t = A_mul(g, tau, z)
            omega = vdot(t, s) / vdot(t, t)
            x = x + alpha * y + omega * z
            r = s - omega * t
            if np.sqrt(vdot(r, r).real) <= p.rtol * nb:
                break
        c = x
    q.put((rank, plan.lo, plan.hi, owned(c)))
    dist.barrier()
    dist.destroy_process_group()


def test_slab_plan_arithmetic():
    from paper_2512_21697_b200 import sharding
    p = _make_problem()
    for world in (1, 2, 3, 5):
        plans = sharding.plan_slabs(p, world)
        bounds = sharding.slab_bounds(p.n_ang, world)
        assert bounds[0] == 0 and bounds[-1] == p.n_ang and all(b1 > b0 for b0, b1 in zip(bounds, bounds[1:]))
        assert max(np.diff(bounds)) - min(np.diff(bounds)) <= 1
        covered = np.zeros(p.n_ang, dtype=int)
        for pl in plans:
            covered[pl.lo:pl.hi] += 1
            assert pl.halo_lo == max(0, pl.lo - pl.reach) and pl.halo_hi == min(p.n_ang, pl.hi + pl.reach)
            need = np.zeros(p.n_ang, dtype=int)
            for r, a, b in pl.needs_from(bounds):
                assert bounds[r] <= a < b <= bounds[r + 1]
                need[a:b] += 1
            halo = np.zeros(p.n_ang, dtype=int)
            halo[pl.halo_lo:pl.lo] = 1
            halo[pl.hi:pl.halo_hi] = 1
            assert np.array_equal(need, halo)                       # every halo channel comes from exactly one owner
            loc = sharding.local_problem(p, pl)
            assert loc.n_ang == pl.n_local
            for t, tl in zip(p.terms, loc.terms):                   # owned rows keep all their couplings, halo rows have none
                for a in range(pl.halo_lo, pl.halo_hi):
                    a_loc = a - pl.halo_lo
                    got = set(tl.A_col[tl.A_rowptr[a_loc]:tl.A_rowptr[a_loc + 1]] + pl.halo_lo)
                    want = set(t.A_col[t.A_rowptr[a]:t.A_rowptr[a + 1]]) if pl.lo <= a < pl.hi else set()
                    assert got == want
        assert np.all(covered == 1)
    assert sharding.coupling_reach(p) == 3                           # offsets +-1..+-(L+1), L = 0..2


def test_sharded_cn_step_equals_unsharded_oracle_gloo_world2():
    from oracle import tdde_oracle as orc
    p = _make_problem()
    ops, fact = orc.assemble(p), orc.factor_precond(p)
    c_ref, infos = orc.propagate(p, ops, fact, p.c0, p.n_steps)
    assert max(i.half_iters for i in infos) >= 3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29547, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    res = [q.get(timeout=300) for _ in procs]
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    C = np.zeros((p.n_ang, p.n_rad), dtype=np.complex128)
    for rank, lo, hi, slab in res:
        C[lo:hi] = slab.reshape(hi - lo, p.n_rad)
    assert np.linalg.norm(C.reshape(-1) - c_ref) <= 1e-10 * np.linalg.norm(c_ref)


def test_shard_specs_are_symmetric_and_cover_the_halos():
    """The exchange lists handed to tdde_group_create: every halo channel of every rank is received exactly once from its owner's
    owned slab, and each receive has the matching send on the owner (NCCL pairs them by peer)."""
    import tdde_inputs
    from paper_2512_21697_b200 import sharding
    for n_ang, T, world in [(23, 3, 2), (64, 7, 4), (150, 7, 3), (40, 5, 1)]:
        p = tdde_inputs.make_synthetic(name="spec", n_ang=n_ang, n_r=6, bandwidth=7, n_terms=T, dt=0.01, n_steps=1, rtol=1e-10, seed=1,
                                       with_c0=False)
        parts = sharding.shard_specs(p, world)
        for plan, pl, sp in parts:
            assert pl.n_ang == plan.n_local and sp["own_hi"] - sp["own_lo"] == plan.hi - plan.lo
            covered = np.zeros(plan.n_local, dtype=int)
            covered[sp["own_lo"]:sp["own_hi"]] += 1
            for r, lo, src_lo, n in zip(sp["recv_rank"], sp["recv_lo"], sp["recv_src_lo"], sp["recv_n"]):
                covered[lo:lo + n] += 1
                oplan, _, osp = parts[r]
                assert osp["own_lo"] <= src_lo and src_lo + n <= osp["own_hi"]                 # inside the owner's owned slab
                assert lo + plan.halo_lo == src_lo + oplan.halo_lo                             # the same global channels
                assert (plan.rank, src_lo, n) in list(zip(osp["send_rank"], osp["send_lo"], osp["send_n"]))
            assert np.all(covered == 1)
            # owned rows keep all their couplings, halo rows have none
            for t_loc, t in zip(pl.terms, p.terms):
                cnt = np.diff(t_loc.A_rowptr)
                assert np.all(cnt[:sp["own_lo"]] == 0) and np.all(cnt[sp["own_hi"]:] == 0)
                assert np.array_equal(cnt[sp["own_lo"]:sp["own_hi"]], np.diff(t.A_rowptr)[plan.lo:plan.hi])
