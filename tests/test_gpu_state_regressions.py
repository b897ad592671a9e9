"""Host-side bookkeeping of the context against what the device really holds: sequences of calls in which the library has to
know for which (theta, MAC) the fp32 walk records were written, and whether acc_pot is in the order of the particles.
Each sequence ends in a comparison with the oracle (counts bit for bit, forces in tolerance) or with a second context that
takes the plain path."""
import numpy as np
import pytest
import torch

import bh_inputs
import oracle
from parity_common import check_forces, compare_counts, export_numpy, gpu_tree
from test_gpu_blockstep import _block_pair, _check_block_step

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def BH():
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import BarnesHut
    return BarnesHut


def test_theta_changes_between_block_steps(BH):
    """A block step refreshes the moments (and the walk records) of the cells above the active particles only.  With another
    theta than the records of the other cells were written for, all of them have to be redone: the counts are the oracle's
    for the new theta, not a mixture."""
    n = 20000
    bh, bs, theta, eps = _block_pair(BH, n, 211, 5, 0.15)
    bs, _ = _check_block_step(bh, bs, theta, eps)
    partial_at_a_change = 0
    last = theta
    for th in (0.45, 0.8, 0.8, theta, 0.5, theta):
        bs, b = _check_block_step(bh, bs, th, eps)
        partial_at_a_change += int(th != last and int(b["stats"].n_active) < n)
        last = th
    assert partial_at_a_change >= 2                       # (a step that moves everybody refreshes every cell anyway)


def test_mac_changes_before_a_partial_refresh(BH):
    """bh_set_mac, then a refresh of the cells above a few particles, then a full walk: every cell's opening radius is the
    new criterion's (oracle counts for the minimum-distance MAC), and back again."""
    n = 20000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=223)
    theta, eps = prm["theta"], prm["eps"]
    bh = BH(n)
    gpu_tree(bh, pm, vel, theta, eps)
    st = oracle.tree_build(pm, vel)
    active = torch.zeros(n, dtype=torch.uint8, device="cuda")
    active[::997] = 1
    for mac in (1, 0):
        bh.set_mac(mac)
        bh.refresh_moments_active(active)                 # positions unchanged: the moments stay, the records are rewritten where dirty
        bh.compute_forces(theta, eps)
        g = export_numpy(bh)
        oracle.compute_forces(st, theta, eps, mac_kind=mac)
        assert np.array_equal(g["cell_r2open"], st.mac[:, 2])
        bad = compare_counts(g, st)
        assert not bad, f"mac {mac}:\n" + "\n".join(bad)
        check_forces(g, st)


def test_graph_replays_between_walks_at_another_theta(BH):
    """The captured step writes the walk records for ITS theta; a plain bh_compute_forces at another theta before and after
    a replay must notice that (and the capture itself, which runs nothing, must not pretend the records changed)."""
    n = 20000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=227)
    eps, dt = prm["eps"], prm["dt"]
    a, b = BH(n), BH(n)
    gpu_tree(a, pm, vel, 0.7, eps)
    gpu_tree(b, pm, vel, 0.7, eps)
    b.step_graph_build(0.5, eps, dt)                      # nothing runs: the device still holds the records for 0.7 ...
    a.compute_forces(0.5, eps)
    b.compute_forces(0.5, eps)                            # ... so this walk has to rewrite them
    ga, gb = export_numpy(a), export_numpy(b)
    for k in ("group_npc", "group_npp", "cell_r2open", "acc_pot"):
        assert np.array_equal(ga[k], gb[k]), k
    st = oracle.compute_forces(oracle.tree_build(pm, vel), 0.5, eps)
    assert not compare_counts(gb, st)
    for _ in range(2):
        a.compute_forces(0.7, eps); b.compute_forces(0.7, eps)
        a.leapfrog_step(0.5, eps, dt); b.step_graph_launch()           # records are now for 0.5 on both
        a.compute_forces(0.7, eps); b.compute_forces(0.7, eps)         # and must be redone for 0.7
        ga, gb = export_numpy(a), export_numpy(b)
        for k in ("pos_mass", "vel", "group_npc", "group_npp", "cell_r2open", "acc_pot"):
            assert np.array_equal(ga[k], gb[k]), k
        st = oracle.compute_forces(oracle.tree_build(ga["pos_mass"].copy(), ga["vel"].copy(), ga["id"].view(np.uint32).copy()), 0.7, eps)
        assert np.array_equal(gb["cell_r2open"], st.mac[:, 2]) and not compare_counts(gb, st)
    out = np.empty((n, 4), np.float32)
    b.get_particles(acc_pot=out)                          # a replay is a full walk: acc_pot is in order
    torch.cuda.synchronize()
    assert np.array_equal(out, gb["acc_pot"])


def test_acc_pot_after_a_rebuild_and_an_active_walk(BH):
    """bh_tree_build re-sorts the particles; an active-subset walk afterwards writes some rows of acc_pot only, so the others
    still belong to other particles: reading acc_pot is refused.  bh_block_step with a rebuild moves the held accelerations
    into place first, so there every row belongs to its particle."""
    from paper_1106_1900_b200 import BhError
    n = 15000
    bh, bs, theta, eps = _block_pair(BH, n, 229, 3, 0.2)
    bs, _ = _check_block_step(bh, bs, theta, eps)
    bs, b = _check_block_step(bh, bs, theta, eps, rebuild=True)
    out = np.empty((n, 4), np.float32)
    bh.get_particles(acc_pot=out)
    torch.cuda.synchronize()
    gb = bs.tree.gbegin.astype(np.int64)
    walked = np.repeat(np.add.reduceat(b["active"].astype(np.int64), gb) > 0, bs.tree.gcount)
    act = b["active"].astype(bool)
    assert 0 < walked.sum() < n
    assert np.array_equal(out[~walked], b["acc_held"][~walked])        # not walked: the held acceleration of THIS particle
    assert np.array_equal(out[act], b["acc_held"][act])                # active: the new one (the corrector holds it now)
    # the same without the block scheme: build, then a walk of a subset only
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=233)
    c = BH(n)
    gpu_tree(c, pm, vel, theta, eps)
    c.kick_drift(0.0, 1.0 / 64)
    c.tree_build()
    flags = torch.zeros(n, dtype=torch.uint8, device="cuda")
    flags[: n // 10] = 1
    c.compute_forces_active(theta, eps, flags)
    with pytest.raises(BhError):
        c.get_particles(acc_pot=out)
    c.compute_forces(theta, eps)
    c.get_particles(acc_pot=out)                                       # a full walk puts every row in order


def test_block_step_leaves_the_sort_counters_alone(BH):
    """bh_stats.sort_passes / sort_retries describe the last build; a block step without a rebuild does not touch them."""
    bh, bs, theta, eps = _block_pair(BH, 20000, 239, 3, 0.2)
    s0 = bh.sync_status()
    assert 0 < s0.sort_passes <= 8
    bh.block_step(theta, eps)
    s1 = bh.sync_status()
    assert s1.sort_passes == s0.sort_passes and s1.sort_retries == s0.sort_retries


def test_tick_counter_end_is_reported(BH):
    """32-bit ticks: with max_rung = 20 and every particle on the longest step a block step advances 2^20 ticks; the deferred
    status turns BH_ERR_STATE when less than two longest steps are left, and not before."""
    n = 512
    pm, vel, _ = bh_inputs.make("c1", n=n, seed=241)
    bh = BH(n)
    gpu_tree(bh, pm, vel, 0.7, 0.05)
    bh.block_init(0.05, 1e9, 1e-7, 20)                    # eta huge: rung 0 for everybody; dt tiny: nothing really moves
    for _ in range(4093):
        bh.block_step(0.7, 0.05)
    assert bh.sync_status(check=False).status == 0
    assert int(bh.block_state(arrays=False)["stats"].now_tick) == 4093 << 20
    bh.block_step(0.7, 0.05)
    assert bh.sync_status(check=False).status == -3
    b = bh.block_state()
    assert int(b["stats"].now_tick) == 4094 << 20 and np.all(b["tick"] == 4094 << 20)   # the step itself is still exact
