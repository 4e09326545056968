"""Channel-slab sharding plan (SURVEY.md 8(f) NEXT-3; PAPER.md:279-297 section 3.2, :307 section 3.3) -- the host side.

The paper partitions the rows (angular channels) of the coupling matrix among ranks, exchanges the x-slabs of coupled channels
before every operator apply, keeps the block-diagonal preconditioner rank-local and sums every inner product over the ranks.
On NVSwitch the same decomposition is: contiguous channel slabs, halo slabs of +-(coupling reach) channels gathered before each
apply, one all-reduce of 3 partial sums per fused reduction.  This module holds the index arithmetic of that decomposition --
which channels a rank owns, which it must receive, and the rank-local problem (owned rows of every A_L with columns renumbered
into [halo | owned | halo]) that a per-rank `Tdde` handle is created from, and the exchange lists `TddeGroup` (tdde_group_* in
include/tdde.h, csrc/tdde_shard.cu) takes.  It moves no data and computes nothing on vectors.  `tests/test_sharding_gloo.py`
exercises the plan with two gloo ranks on CPU against the unsharded oracle; the device path is tested on one GPU with all shards
in one process (tests/test_gpu_sharding.py).
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import List

import numpy as np


@dataclass
class SlabPlan:
    rank: int
    world: int
    lo: int            # owned channels [lo, hi) (global numbering)
    hi: int
    halo_lo: int       # channels present on the rank: [halo_lo, halo_hi) contains [lo, hi) plus everything its rows couple to
    halo_hi: int
    reach: int         # largest |column - row| over all terms

    @property
    def n_local(self) -> int:
        return self.halo_hi - self.halo_lo

    @property
    def own_slice(self) -> slice:
        """Owned channels in LOCAL numbering."""
        return slice(self.lo - self.halo_lo, self.hi - self.halo_lo)

    def needs_from(self, bounds: List[int]):
        """[(owner rank, global lo, global hi)] of the halo channels this rank must receive before an apply."""
        out = []
        for r in range(self.world):
            if r == self.rank:
                continue
            a, b = max(bounds[r], self.halo_lo), min(bounds[r + 1], self.halo_hi)
            if a < b:
                out.append((r, a, b))
        return out


def slab_bounds(n_ang: int, world: int) -> List[int]:
    """Contiguous, balanced channel slabs: bounds[r] .. bounds[r + 1]."""
    base, rem = divmod(n_ang, world)
    b = [0]
    for r in range(world):
        b.append(b[-1] + base + (1 if r < rem else 0))
    return b


def coupling_reach(problem) -> int:
    reach = 0
    for t in problem.terms:
        rows = np.repeat(np.arange(problem.n_ang), np.diff(t.A_rowptr))
        if len(rows):
            reach = max(reach, int(np.max(np.abs(t.A_col.astype(np.int64) - rows))))
    return reach


def plan_slabs(problem, world: int) -> List[SlabPlan]:
    if world < 1 or world > problem.n_ang:
        raise ValueError("need 1 <= world <= n_ang")
    bounds = slab_bounds(problem.n_ang, world)
    reach = coupling_reach(problem)
    return [SlabPlan(r, world, bounds[r], bounds[r + 1], max(0, bounds[r] - reach), min(problem.n_ang, bounds[r + 1] + reach), reach)
            for r in range(world)]


def local_problem(problem, plan: SlabPlan):
    """The rank-local problem: channels [halo_lo, halo_hi) renumbered from 0; rows of A_L kept for OWNED channels only (halo channels
    are inputs: their outputs belong to another rank), columns shifted by halo_lo.  Blocks (per kappa-class) are shared unchanged."""
    from tdde_inputs import Problem, Term
    n_loc = plan.n_local
    terms = []
    for t in problem.terms:
        rowptr = np.zeros(n_loc + 1, dtype=np.int32)
        cols, vals = [], []
        for a_loc in range(n_loc):
            a = a_loc + plan.halo_lo
            if plan.lo <= a < plan.hi:
                sl = slice(t.A_rowptr[a], t.A_rowptr[a + 1])
                c = t.A_col[sl].astype(np.int64) - plan.halo_lo
                if len(c) and (c.min() < 0 or c.max() >= n_loc):
                    raise AssertionError("coupling leaves the halo: reach too small")
                cols.append(c.astype(np.int32))
                vals.append(t.A_val[sl])
            rowptr[a_loc + 1] = rowptr[a_loc] + (len(cols[-1]) if plan.lo <= a < plan.hi else 0)
        terms.append(Term(w=t.w, R_band=t.R_band, A_rowptr=rowptr,
                          A_col=np.concatenate(cols) if cols else np.zeros(0, np.int32),
                          A_val=np.concatenate(vals) if vals else np.zeros(0, np.complex128)))
    c0 = problem.c0.reshape(problem.n_ang, problem.n_rad)[plan.halo_lo:plan.halo_hi].reshape(-1).copy() if problem.c0.size else problem.c0
    return replace(problem, name=f"{problem.name}-rank{plan.rank}", n_ang=n_loc, cls_of_chan=problem.cls_of_chan[plan.halo_lo:plan.halo_hi].copy(),
                   terms=terms, c0=c0)


def shard_specs(problem, world: int):
    """[(plan, local problem, spec)] per rank; spec = the exchange lists of tdde_shard in LOCAL channel numbering:
    recv: halo piece [recv_lo, recv_lo + n) of this rank = channels [recv_src_lo, ...) of rank recv_rank (local numbering there);
    send: owned piece [send_lo, send_lo + n) of this rank goes to rank send_rank."""
    plans = plan_slabs(problem, world)
    bounds = slab_bounds(problem.n_ang, world)
    out = []
    for pl in plans:
        spec = {"rank": pl.rank, "world": world, "own_lo": pl.lo - pl.halo_lo, "own_hi": pl.hi - pl.halo_lo,
                "recv_rank": [], "recv_lo": [], "recv_src_lo": [], "recv_n": [], "send_rank": [], "send_lo": [], "send_n": []}
        for owner, a, b in pl.needs_from(bounds):
            spec["recv_rank"].append(owner)
            spec["recv_lo"].append(a - pl.halo_lo)
            spec["recv_src_lo"].append(a - plans[owner].halo_lo)
            spec["recv_n"].append(b - a)
        for other in plans:
            if other.rank == pl.rank:
                continue
            for owner, a, b in other.needs_from(bounds):
                if owner == pl.rank:
                    spec["send_rank"].append(other.rank)
                    spec["send_lo"].append(a - pl.halo_lo)
                    spec["send_n"].append(b - a)
        out.append((pl, local_problem(problem, pl), spec))
    return out
