"""Group-sharded walk over several GPUs of one node ("each thread block executes the
same algorithm but on a different set of particles", L268 for the cluster outlook).

Every rank holds ALL particles and builds the identical tree (S0-S6 are ~15 % of a step); rank r walks and evaluates only
the groups that hold a particle of its contiguous share of the key-sorted order (bh_compute_forces_active), keeps the
rows of its share, and ONE all-reduce (sum with zeros = exact) of the acc_pot array gives every rank every force; the
kicks and the drift are then done redundantly, so the ranks stay bit-identical without ever exchanging positions.
One process per GPU; `torch.distributed` (NCCL over NVLink on GPUs) is the only plumbing; this module only marshals.

A step is bit-identical to BarnesHut.leapfrog_step on one GPU as long as no group is deferred to the fused kernel
(per-group sums do not depend on which other groups are walked).
"""
from __future__ import annotations

import torch

from .binding import BarnesHut


def share_bounds(n: int, world: int) -> list[int]:
    """Particle index boundaries of the ranks' shares of the sorted order: rank r owns [b[r], b[r+1])."""
    return [(n * r) // world for r in range(world + 1)]


def share_mask(n: int, world: int, rank: int, device) -> torch.Tensor:
    """uint8[n]: 1 on this rank's share.  A group that straddles a boundary is walked by both neighbours (identical values);
    each keeps the rows of its own share."""
    b = share_bounds(n, world)
    m = torch.zeros(n, dtype=torch.uint8, device=device)
    m[b[rank]: b[rank + 1]] = 1
    return m


def keep_own_rows(acc: torch.Tensor, n: int, world: int, rank: int) -> torch.Tensor:
    """Zero the rows of the other ranks' shares in place (what the all-reduce then fills in)."""
    b = share_bounds(n, world)
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

    def set_particles(self, pos_mass, vel=None, ids=None):
        """The SAME particles on every rank."""
        self.bh.set_particles(pos_mass, vel, ids)
        self.mask = share_mask(self.bh.n, self.world, self.rank, self.bh.device)

    def compute_forces(self, theta: float, eps: float):
        """S7 + S8 of this rank's share, then the exchange: afterwards every rank holds every particle's acc_pot."""
        bh = self.bh
        if self.world == 1:
            bh.compute_forces(theta, eps)
            return
        bh.compute_forces_active(theta, eps, self.mask)
        acc = bh.acc_view()
        keep_own_rows(acc, bh.n, self.world, self.rank)
        self.dist.all_reduce(acc, op=self.dist.ReduceOp.SUM, group=self.group)

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
