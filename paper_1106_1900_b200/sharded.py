"""Group-sharded walk over several GPUs of one node ("each thread block executes the
same algorithm but on a different set of particles", L268 for the cluster outlook).

Every rank holds ALL particles and builds the identical tree (S0-S6 are ~15 % of a step); rank r walks and evaluates only
the groups that hold a particle of its contiguous share of the key-sorted order (bh_compute_forces_active), keeps the
rows of its share, and ONE all-reduce (sum with zeros = exact) of the acc_pot array gives every rank every force; the
kicks and the drift are then done redundantly, so the ranks stay bit-identical without ever exchanging positions.
One process per GPU; `torch.distributed` (NCCL over NVLink on GPUs) is the only plumbing; this module only marshals.

A step is bit-identical to BarnesHut.leapfrog_step on one GPU as long as no group is deferred to the fused kernel
(per-group sums do not depend on which other groups are walked).

Shares: the first force evaluation splits the key-sorted particles into equal counts; afterwards the boundaries follow the
WORK of the previous evaluation, sum over groups of n_g (20 n_pp + 64 n_pc), so that every rank gets
the same number of flops rather than of particles (the core of a Plummer sphere costs several times the halo).  The
per-group work of the ranks is combined by a second, small all-reduce (8 bytes per group); every rank derives the same
boundaries from it.  Particles move little between rebuilds, so last step's boundaries (as positions in the sorted
order) fit the next step's groups.
"""
from __future__ import annotations

import torch

from .binding import BarnesHut


def share_bounds(n: int, world: int) -> list[int]:
    """Particle index boundaries of the ranks' shares of the sorted order: rank r owns [b[r], b[r+1])."""
    return [(n * r) // world for r in range(world + 1)]


def balanced_bounds(group_begin: torch.Tensor, work: torch.Tensor, n: int, world: int) -> list[int]:
    """Boundaries that give every rank the same WORK: group_begin int[G] (first particle of each group, ascending), work[G]
    (flops of each group in the last walk).  Rank r starts at the first group whose preceding work reaches r / world of
    the total; boundaries are group starts, strictly increasing wherever there are enough groups."""
    gb = group_begin.to(torch.int64).cpu()
    w = work.to(torch.float64).cpu()
    G = int(gb.numel())
    if G == 0 or float(w.sum()) <= 0.0:
        return share_bounds(n, world)
    before = torch.cumsum(w, 0) - w                      # work of the groups before each group
    total = float(w.sum())
    b = [0]
    for r in range(1, world):
        g = int(torch.searchsorted(before, torch.tensor(total * r / world, dtype=torch.float64), right=False))
        g = min(max(g, 1), G - 1) if G > 1 else 0
        b.append(max(int(gb[g]), b[-1]))
    b.append(n)
    return b


def share_mask(n: int, world: int, rank: int, device, bounds: list[int] | None = None) -> torch.Tensor:
    """uint8[n]: 1 on this rank's share.  A group that straddles a boundary is walked by both neighbours (identical values);
    each keeps the rows of its own share."""
    b = share_bounds(n, world) if bounds is None else bounds
    m = torch.zeros(n, dtype=torch.uint8, device=device)
    m[b[rank]: b[rank + 1]] = 1
    return m


def keep_own_rows(acc: torch.Tensor, n: int, world: int, rank: int, bounds: list[int] | None = None) -> torch.Tensor:
    """Zero the rows of the other ranks' shares in place (what the all-reduce then fills in)."""
    b = share_bounds(n, world) if bounds is None else bounds
    acc[: b[rank]].zero_()
    acc[b[rank + 1]:].zero_()
    return acc


class ShardedBarnesHut:
    """The calls of BarnesHut, with the walk of a step shared by the ranks of a torch.distributed process group."""

    def __init__(self, n_max: int, group=None, **cfg):
        import torch.distributed as dist
        self.dist = dist
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.bh = BarnesHut(n_max, **cfg)
        self.mask = None
        self.bounds = None           # particle index boundaries of the shares (positions in the key-sorted order)
        self.balance = True          # False: equal particle counts every step
        self.last_work = None        # flops per rank of the last evaluation (after the exchange), for reporting

    def set_particles(self, pos_mass, vel=None, ids=None):
        """The SAME particles on every rank."""
        self.bh.set_particles(pos_mass, vel, ids)
        self.bounds = share_bounds(self.bh.n, self.world)
        self.mask = share_mask(self.bh.n, self.world, self.rank, self.bh.device, self.bounds)

    def compute_forces(self, theta: float, eps: float):
        """S7 + S8 of this rank's share, then the exchange: afterwards every rank holds every particle's acc_pot."""
        bh = self.bh
        if self.world == 1:
            bh.compute_forces(theta, eps)
            return
        bh.compute_forces_active(theta, eps, self.mask)
        acc = bh.acc_view()
        keep_own_rows(acc, bh.n, self.world, self.rank, self.bounds)
        self.dist.all_reduce(acc, op=self.dist.ReduceOp.SUM, group=self.group)
        if self.balance:
            # the work of every group (each rank knows its own groups; a group walked by two neighbours counts once: MAX)
            gb, npc, npp = bh.group_views()
            ng = (gb[1:] - gb[:-1]).to(torch.int64)
            work = ng * (20 * npp.to(torch.int64) + 64 * npc.to(torch.int64))
            self.dist.all_reduce(work, op=self.dist.ReduceOp.MAX, group=self.group)
            cum = torch.cumsum(work, 0)
            idx = torch.searchsorted(gb[:-1].to(torch.int64), torch.tensor(self.bounds[1:-1], device=gb.device, dtype=torch.int64), right=False)
            edges = torch.cat([torch.zeros(1, dtype=torch.int64, device=gb.device), cum[(idx - 1).clamp(min=0)], cum[-1:]])
            self.last_work = (edges[1:] - edges[:-1]).tolist()
            self.bounds = balanced_bounds(gb[:-1], work, bh.n, self.world)
            self.mask = share_mask(bh.n, self.world, self.rank, bh.device, self.bounds)

    def tree_build(self):
        self.bh.tree_build()

    def leapfrog_step(self, theta: float, eps: float, dt: float):
        """kick(dt/2) + drift(dt), S0-S6 (redundant), this rank's share of S7 + S8, all-reduce, kick(dt/2)."""
        bh = self.bh
        h = 0.5 * dt
        bh.kick_drift(h, dt)
        bh.tree_build()
        self.compute_forces(theta, eps)
        bh.kick_drift(h, 0.0)            # a pure kick: positions, tree and forces stay valid

    def __getattr__(self, name):         # sync_status, export_tree, get_particles, ... : the underlying context's
        return getattr(self.bh, name)
