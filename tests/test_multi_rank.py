"""Host-side logic of the N > 1 path of bench.py, on CPU with the gloo backend and world size 2 (no GPU).

DESIGN.md section 9: replicas only -- each rank steps its own replica (its own seed), no data-path collective; the
job's time is the slowest rank's (all-reduce MAX of one scalar); rank 0 alone reports; the reference arm runs on
rank 0 only.  The ranks here also run the oracle on their replica to show the replicas really differ.
"""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np
    import torch.distributed as dist
    import bench, bh_inputs, oracle
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    pm, vel, prm = bench._make_inputs("c1", 2048, rank)
    st = oracle.tree_build(pm, vel)
    local_ms = 10.0 * (rank + 1)                        # rank 1 is the slow one
    total_ms = bench.max_over_ranks(local_ms, world)
    value = bench.job_throughput(world, 2048, 4, total_ms * 1e-3)
    out = dict(rank=rank, seed=bench.rank_seed("c1", rank), checksum=float(np.float64(pm[:, :3]).sum()),
               cells=st.tree.ncells, total_ms=total_ms, value=value)
    print("RANKOUT " + json.dumps(out), flush=True)
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def test_two_ranks_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29731", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    import re
    # the two ranks share one pipe: their lines may arrive glued together, so cut at the marker, not at newlines
    outs = sorted((json.loads(m) for m in re.findall(r"RANKOUT (\{[^{}]*\})", r.stdout)), key=lambda o: o["rank"])
    assert [o["rank"] for o in outs] == [0, 1]
    assert outs[0]["seed"] != outs[1]["seed"] and outs[0]["checksum"] != outs[1]["checksum"]      # different replicas
    assert outs[0]["total_ms"] == outs[1]["total_ms"] == 20.0                                      # max over ranks
    assert outs[0]["value"] == 2 * 2048 * 4 / 20e-3                                                 # whole-job aggregate


SHARD_WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np, torch
    import torch.distributed as dist
    import bh_inputs, oracle
    from paper_1106_1900_b200.sharded import keep_own_rows, share_bounds, share_mask
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    n = 3000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=71)             # the SAME particles on every rank
    st = oracle.tree_build(pm, vel)
    t = st.tree
    mask = share_mask(n, world, rank, "cpu").numpy()
    sel = np.array([g for g in range(t.ngroups) if mask[t.gbegin[g]: t.gbegin[g] + t.gcount[g]].any()], np.int64)
    oracle.compute_forces(st, prm["theta"], prm["eps"], sel=sel)   # this rank's share of the walk (the oracle stands in for the GPU)
    acc = torch.from_numpy(np.nan_to_num(st.accpot))
    keep_own_rows(acc, n, world, rank)
    dist.all_reduce(acc, op=dist.ReduceOp.SUM)                     # the one exchange of a step
    full = oracle.compute_forces(oracle.tree_build(pm, vel), prm["theta"], prm["eps"]).accpot
    out = dict(rank=rank, groups=int(sel.size), all_groups=int(t.ngroups), equal=bool(np.array_equal(acc.numpy(), full)),
               bounds=share_bounds(n, world))
    print("RANKOUT " + json.dumps(out), flush=True)
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def test_group_sharded_walk_two_ranks_gloo(tmp_path):
    """Host logic of the sharded walk (shares, own rows, one all-reduce) with the oracle as the force provider."""
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29733", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    import re
    outs = sorted((json.loads(m) for m in re.findall(r"RANKOUT (\{[^{}]*\})", r.stdout)), key=lambda o: o["rank"])
    assert [o["rank"] for o in outs] == [0, 1]
    assert all(o["equal"] for o in outs)                                   # every rank ends with every force, bit for bit
    G = outs[0]["all_groups"]
    assert G <= outs[0]["groups"] + outs[1]["groups"] <= G + 1             # at most the straddling group is walked twice
    assert outs[0]["bounds"] == [0, 1500, 3000]


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "c1"], capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == ""          # other ranks exit 0 without work
    env["RANK"] = "0"
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0", "--config", "c1"], capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    import json
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "particles/s"


def test_bench_starts_its_own_ranks_without_torchrun():
    """`python bench.py --gpus 2` with no launcher must create two ranks itself (dry run: process group + max-over-ranks only)."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run-ranks"], capture_output=True, text=True,
                       timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["max_over_ranks"] == 2.0


BALANCE_WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np, torch
    import torch.distributed as dist
    import bh_inputs, oracle
    from paper_1106_1900_b200.sharded import balanced_bounds, keep_own_rows, share_bounds, share_mask
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    n = 6000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=73)
    st = oracle.tree_build(pm, vel)
    t = st.tree
    full = oracle.compute_forces(oracle.tree_build(pm, vel), prm["theta"], prm["eps"])
    work_all = t.gcount * (20 * full.npp + 64 * full.npc)
    bounds = share_bounds(n, world)
    imb = []
    for it in range(2):                                             # equal counts first, then balanced by the measured work
        mask = share_mask(n, world, rank, "cpu", bounds).numpy()
        sel = np.array([g for g in range(t.ngroups) if mask[t.gbegin[g]: t.gbegin[g] + t.gcount[g]].any()], np.int64)
        oracle.compute_forces(st, prm["theta"], prm["eps"], sel=sel)
        acc = torch.from_numpy(np.nan_to_num(st.accpot))
        keep_own_rows(acc, n, world, rank, bounds)
        dist.all_reduce(acc, op=dist.ReduceOp.SUM)
        work = torch.zeros(t.ngroups, dtype=torch.int64)
        work[sel] = torch.from_numpy(t.gcount[sel] * (20 * st.npp[sel] + 64 * st.npc[sel]))
        mine = float(work.sum())
        dist.all_reduce(work, op=dist.ReduceOp.MAX)
        per = torch.tensor([mine], dtype=torch.float64); allw = [torch.zeros(1, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(allw, per)
        imb.append(max(float(x) for x in allw) * world / float(work.sum()))
        equal = bool(np.array_equal(acc.numpy(), full.accpot))
        bounds = balanced_bounds(torch.from_numpy(t.gbegin), work, n, world)
    out = dict(rank=rank, imbalance=imb, equal=equal, bounds=bounds, work_ok=bool(np.array_equal(work.numpy(), work_all)))
    print("RANKOUT " + json.dumps(out), flush=True)
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def test_balanced_shares_two_ranks_gloo(tmp_path):
    """Shares by the previous walk's flops per group: same forces, and the slowest rank's work drops."""
    script = tmp_path / "balance_worker.py"
    script.write_text(BALANCE_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29735", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    import re
    outs = sorted((json.loads(m) for m in re.findall(r"RANKOUT (\{[^{}]*\})", r.stdout)), key=lambda o: o["rank"])
    assert [o["rank"] for o in outs] == [0, 1]
    assert all(o["equal"] and o["work_ok"] for o in outs)
    assert outs[0]["bounds"] == outs[1]["bounds"] and outs[0]["bounds"][1] != 3000        # every rank derives the same, moved boundary
    assert outs[0]["imbalance"][1] < outs[0]["imbalance"][0] and outs[0]["imbalance"][1] < 1.1, outs[0]["imbalance"]
