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


TWO_RANK_WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
sys.path.insert(0, os.path.join(%r, "tests"))
import numpy as np, torch
import torch.distributed as dist
import bh_inputs, oracle
from parity_common import check_forces, compare_counts, compare_tree, export_numpy
from paper_1106_1900_b200 import ShardedBarnesHut
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(0)                       # both ranks share the one GPU of the box; their kernels never wait for each other,
dist.init_process_group("gloo")                # the exchange goes through gloo (NCCL refuses two ranks on one device)
n = 20000
pm, vel, prm = bh_inputs.make("c1", n=n, seed=79)
theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
bh = ShardedBarnesHut(n)
assert bh.world == 2
bh.set_particles(pm, vel)
b0 = list(bh.bounds)                           # equal particle counts before the first evaluation
bh.tree_build()
bh.compute_forces(theta, eps)                  # world > 1: own share by bh_compute_forces_active, all-reduce of acc_pot, work all-reduce
st = oracle.compute_forces(oracle.tree_build(pm, vel), theta, eps)
g = export_numpy(bh)
bad = compare_tree(g, st)
mine = np.nonzero(g["group_npc"] + g["group_npp"] > 0)[0]      # the groups this rank walked
compare_counts(g, st, sel=mine, problems=bad)
assert not bad, bad
e0 = check_forces(g, st)                       # EVERY particle's force is present on EVERY rank, within the tolerance of the oracle
for step in range(2):
    so = oracle.tree_build(g["pos_mass"].copy(), g["vel"].copy(), g["id"].view(np.uint32).copy())
    so.accpot = g["acc_pot"].astype(np.float64)
    s2 = oracle.leapfrog_step(so, theta, eps, dt)
    bh.leapfrog_step(theta, eps, dt)
    g = export_numpy(bh)
    bad = compare_tree(g, s2, check_vel=False)
    assert not bad, bad
    check_forces(g, s2)
torch.cuda.synchronize()
out = dict(rank=rank, groups_walked=int(mine.size), groups=int(g["n_groups"]), acc_rms=e0["acc_rms"], bounds0=b0, bounds=list(bh.bounds),
           work=bh.last_work, checksum=float(np.float64(g["acc_pot"]).sum()))
print("RANKOUT " + json.dumps(out), flush=True)
dist.barrier()
dist.destroy_process_group()
"""


def test_two_ranks_share_the_walk_and_match_the_oracle(tmp_path):
    """ShardedBarnesHut with world size 2 for real: two processes (on the one GPU), redundant build, each walks its share,
    the all-reduce delivers every force to both; checked against the ORACLE per call, and the shares move to balance flops."""
    import json
    import os
    import re
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "two_rank_worker.py"
    script.write_text(TWO_RANK_WORKER % (root, root))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29741", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    outs = sorted((json.loads(m) for m in re.findall(r"RANKOUT (\{[^{}]*\})", r.stdout)), key=lambda o: o["rank"])
    assert [o["rank"] for o in outs] == [0, 1]
    G = outs[0]["groups"]
    assert outs[0]["checksum"] == outs[1]["checksum"]                          # the ranks stay bit-identical
    assert outs[0]["bounds0"] == [0, 10000, 20000] and outs[0]["bounds"] == outs[1]["bounds"] and outs[0]["bounds"][1] != 10000
    w = outs[0]["work"]
    assert max(w) / (sum(w) / 2) < 1.15, w                                     # balanced by the previous step's flops
