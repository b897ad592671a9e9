"""Group-sharded walk: the one-rank degenerate case against the plain step, and the shares of three
ranks computed one after the other on one GPU (no process waits for another) against the walk of all groups."""
import numpy as np
import pytest
import torch

import bh_inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mod():
    import __graft_entry__ as g
    g.build()
    import paper_1106_1900_b200 as m
    return m


def test_one_rank_step_is_the_plain_step(mod):
    pm, vel, prm = bh_inputs.make("c1", n=12000, seed=61)
    a, b = mod.BarnesHut(12000), mod.ShardedBarnesHut(12000)
    out = []
    for bh in (a, b):
        bh.set_particles(pm, vel)
        bh.tree_build()
        bh.compute_forces(prm["theta"], prm["eps"])
        for _ in range(3):
            bh.leapfrog_step(prm["theta"], prm["eps"], prm["dt"])
        p, v, f = (np.empty((12000, 4), np.float32) for _ in range(3))
        bh.get_particles(p, v, f)
        torch.cuda.synchronize()
        out.append((p, v, f))
    for x, y in zip(*out):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("world", [2, 3])
def test_shares_add_up_to_the_walk_of_all_groups(mod, world):
    n = 20000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=67)
    full = mod.BarnesHut(n)
    full.set_particles(pm, vel); full.tree_build(); full.compute_forces(prm["theta"], prm["eps"])
    ref = full.export_tree()
    acc_ref = ref["acc_pot"].clone()
    total = torch.zeros_like(acc_ref)
    npc = torch.zeros_like(ref["group_npc"])
    walked = 0
    for rank in range(world):
        bh = mod.BarnesHut(n)
        bh.set_particles(pm, vel); bh.tree_build()
        bh.compute_forces_active(prm["theta"], prm["eps"], mod.share_mask(n, world, rank, bh.device))
        acc = bh.acc_view()
        torch.cuda.synchronize()
        total += mod.keep_own_rows(acc.clone(), n, world, rank)          # (the all-reduce of the real thing)
        t = bh.export_tree()
        npc = torch.maximum(npc, t["group_npc"])
        walked += int((t["group_npc"] + t["group_npp"] > 0).sum())
    assert torch.equal(total, acc_ref)                                    # bit-identical: per-group sums do not depend on the subset
    assert torch.equal(npc, ref["group_npc"])
    G = int(ref["n_groups"])
    assert G <= walked <= G + world - 1                                   # only groups that straddle a boundary are walked twice
    b = mod.share_bounds(n, world)
    assert b[0] == 0 and b[-1] == n and all(x < y for x, y in zip(b, b[1:]))
