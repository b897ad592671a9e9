"""bh_step_graph_build / bh_step_graph_launch: a step captured into a CUDA graph and replayed (include/bh.h promises that the
hot calls only enqueue work) -- per-call parity with the oracle, and bit-identity with plain bh_leapfrog_step launches."""
import numpy as np
import pytest

import bh_inputs
import oracle
from parity_common import check_forces, compare_counts, compare_tree, export_numpy, gpu_tree

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def BH():
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import BarnesHut
    return BarnesHut


@pytest.mark.parametrize("front_mode", [0, 1])
def test_replayed_step_tracks_the_oracle(BH, front_mode):
    pm, vel, prm = bh_inputs.make("c1")
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    bh = BH(pm.shape[0], front_mode=front_mode)
    g = gpu_tree(bh, pm, vel, theta, eps)
    bh.set_stage_timing(True)
    bh.step_graph_build(theta, eps, dt)
    for step in range(3):                       # three replays: both parities of the particle buffers
        st = oracle.tree_build(g["pos_mass"].copy(), g["vel"].copy(), g["id"].view(np.uint32).copy())
        st.accpot = g["acc_pot"].astype(np.float64)
        st2 = oracle.leapfrog_step(st, theta, eps, dt)
        bh.step_graph_launch()
        g = export_numpy(bh)
        bad = compare_tree(g, st2, check_vel=False)
        compare_counts(g, st2, problems=bad)
        assert not bad, f"step {step}:\n" + "\n".join(bad)
        check_forces(g, st2)
        ms = bh.stage_ms()                      # the stage events are part of the graph
        assert ms["sort"] > 0.0 and ms["walk"] > 0.0 and ms["moments"] > 0.0


def test_replay_is_bit_identical_to_plain_launches(BH):
    pm, vel, prm = bh_inputs.make("c1", n=20000, seed=5)
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    a, b = BH(20000), BH(20000)
    gpu_tree(a, pm, vel, theta, eps)
    gpu_tree(b, pm, vel, theta, eps)
    b.step_graph_build(theta, eps, dt)
    for _ in range(4):
        a.leapfrog_step(theta, eps, dt)
        b.step_graph_launch()
    ga, gb = export_numpy(a), export_numpy(b)
    for k in ("pos_mass", "vel", "acc_pot", "id", "key", "group_npc", "group_npp", "cell_mom64"):
        assert np.array_equal(ga[k], gb[k]), k
    assert gb["stats"].launches - ga["stats"].launches == 0      # a replay counts the kernels of the step it stands for


def test_graph_needs_forces_and_survives_new_particles_of_the_same_size(BH):
    from paper_1106_1900_b200 import BhError
    pm, vel, prm = bh_inputs.make("c1", n=3000)
    bh = BH(3000)
    bh.set_particles(pm, vel)
    with pytest.raises(BhError):
        bh.step_graph_build(0.75, 0.01, 0.01)   # no forces yet
    with pytest.raises(BhError):
        bh.step_graph_launch()                   # nothing captured
    g0 = gpu_tree(bh, pm, vel, 0.75, 0.01)
    bh.step_graph_build(0.75, 0.01, 0.01)
    bh.step_graph_launch()
    g1 = export_numpy(bh)
    gpu_tree(bh, pm, vel, 0.75, 0.01)            # same n: the captured step is still valid
    bh.step_graph_launch()
    g2 = export_numpy(bh)
    assert np.array_equal(g1["pos_mass"], g2["pos_mass"]) and np.array_equal(g1["acc_pot"], g2["acc_pot"])
    bh.set_particles(pm[:2000], vel[:2000])
    bh.tree_build(); bh.compute_forces(0.75, 0.01)
    with pytest.raises(BhError):
        bh.step_graph_launch()                   # other n: the graphs were dropped


def test_host_step_pipeline_matches_single_context_steps(BH):
    """HostStepPipeline (two contexts on two streams, copies of one step beside the kernels of the other): every ticket returns
    what the same calls give on one context, bit for bit, whatever the order of completion."""
    import torch
    from paper_1106_1900_b200 import HostStepPipeline
    sets = []
    for k in range(5):
        pm, vel, prm = bh_inputs.make("c1", n=6000, seed=500 + k)
        sets.append((torch.from_numpy(pm).pin_memory(), torch.from_numpy(vel).pin_memory(), torch.arange(6000, dtype=torch.int32).pin_memory()))
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    ref = []
    bh = BH(6000)
    for hp, hv, hid in sets:
        bh.set_particles(hp, hv, hid)
        bh.tree_build()
        bh.compute_forces(theta, eps)
        bh.kick_drift(dt, dt)
        out = (torch.empty((6000, 4)), torch.empty((6000, 4)), torch.empty((6000, 4)), torch.empty(6000, dtype=torch.int32))
        bh.get_particles(*out)
        torch.cuda.synchronize()
        ref.append([o.clone() for o in out])
    bh.close()
    pipe = HostStepPipeline(6000, theta, eps, dt, depth=2)
    tickets = []
    for k, (hp, hv, hid) in enumerate(sets):
        tickets.append(pipe.submit(hp, hv, hid))
        if k >= 1:                                   # read the previous step while this one runs
            got = pipe.result(tickets[k - 1])
            for a, b in zip(got, ref[k - 1]):
                assert torch.equal(a, b)
    got = pipe.result(tickets[-1])
    for a, b in zip(got, ref[-1]):
        assert torch.equal(a, b)
    with pytest.raises(ValueError):
        pipe.result(tickets[0])                      # its buffers have been reused
    pipe.close()
