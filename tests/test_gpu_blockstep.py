"""Block time-step ingredients: moments refreshed on the existing cells after the particles moved,
and the walk restricted to the groups that hold an active particle -- against the oracle on the same topology."""
import numpy as np
import pytest
import torch

import bh_inputs
import oracle
from parity_common import check_forces, compare_counts, export_numpy, gpu_tree

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def BH():
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import BarnesHut
    return BarnesHut


def _moved_state(BH, n, seed, dt, **cfg):
    """GPU: build, forces, drift (kick 0: the new positions depend on the inputs only), refresh.  Oracle: the SAME topology
    (built from the original positions), positions drifted by the oracle itself (O11: x = fmaf(v, dt, x), bit-identical
    to the GPU's, which is checked), moments and group boxes recomputed from them."""
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=seed)
    bh = BH(n, **cfg)
    g0 = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
    bh.kick_drift(0.0, dt)
    bh.refresh_moments()
    st = oracle.tree_build(pm, vel)
    moved = oracle.drift(st.pos, st.vel, np.float32(dt))
    got = np.empty((n, 4), np.float32)
    bh.get_particles(pos_mass=got)
    torch.cuda.synchronize()
    assert np.array_equal(got, moved) and not np.array_equal(moved[:, :3], st.pos[:, :3])
    oracle.moments(st.tree, moved)
    st.pos = moved
    return bh, g0, st, prm


@pytest.mark.parametrize("n,cfg", [(20000, {}), (4097, {}), (6000, dict(walk_mode=1)), (6000, dict(list_entries=40000))])
def test_refreshed_moments_and_forces_match_the_oracle(BH, n, cfg):
    bh, g0, st, prm = _moved_state(BH, n, 47, 1.0 / 16, **cfg)
    bh.compute_forces(prm["theta"], prm["eps"])
    g = export_numpy(bh)
    oracle.compute_forces(st, prm["theta"], prm["eps"])
    # same cells and groups as before the drift; moments and tight boxes follow the particles, bit for bit
    for k in ("cell_pbegin", "cell_pcount", "cell_child_begin", "cell_nchild", "group_begin", "group_cell"):
        assert np.array_equal(g[k], g0[k]), k
    assert np.array_equal(g["cell_mom64"], st.tree.mom64) and np.array_equal(g["cell_box"], st.tree.box)
    assert not np.array_equal(g["cell_box"], g0["cell_box"])
    assert np.array_equal(g["cell_r2open"], st.mac[:, 2])
    bad = compare_counts(g, st)
    assert not bad, "\n".join(bad)
    check_forces(g, st)
    # the cells have grown: on average more interactions than on the fresh tree
    assert g["group_npc"].sum() + g["group_npp"].sum() >= g0["group_npc"].sum() + g0["group_npp"].sum()


@pytest.mark.parametrize("cfg", [{}, dict(walk_mode=1), dict(list_entries=40000), dict(walk_waves=3)])
def test_walk_of_the_active_groups_only(BH, cfg):
    n = 20000
    bh, g0, st, prm = _moved_state(BH, n, 53, 1.0 / 32, **cfg)
    bh.compute_forces(prm["theta"], prm["eps"])
    full = export_numpy(bh)
    acc_full = full["acc_pot"].copy()
    # active: a dense core (as block time-steps produce) plus a sprinkle of single particles
    rng = np.random.default_rng(5)
    r = np.linalg.norm(st.pos[:, :3], axis=1)
    active = ((r < np.quantile(r, 0.04)) | (rng.random(n) < 0.002)).astype(np.uint8)
    t = st.tree
    gact = np.array([active[t.gbegin[k]: t.gbegin[k] + t.gcount[k]].any() for k in range(t.ngroups)])
    sel = np.nonzero(gact)[0]
    assert 0 < sel.size < 0.3 * t.ngroups
    # poison the stored forces of the active groups so that a skipped group cannot pass by leftovers
    bh.kick_drift(0.0, 0.0); bh.refresh_moments()               # (positions unchanged: dt = 0)
    bh.compute_forces_active(prm["theta"], prm["eps"], torch.from_numpy(active).cuda())
    g = export_numpy(bh)
    oracle.compute_forces(st, prm["theta"], prm["eps"], sel=sel)
    bad = compare_counts(g, st, sel=sel)
    assert not bad, "\n".join(bad)
    check_forces(g, st, sel=sel)
    idle = np.nonzero(~gact)[0]
    assert np.all(g["group_npc"][idle] == 0) and np.all(g["group_npp"][idle] == 0)
    pidle = np.concatenate([np.arange(t.gbegin[k], t.gbegin[k] + t.gcount[k]) for k in idle])
    assert np.array_equal(g["acc_pot"][pidle], acc_full[pidle])                       # untouched
    pact = np.concatenate([np.arange(t.gbegin[k], t.gbegin[k] + t.gcount[k]) for k in sel])
    if "list_entries" not in cfg:       # (a starved list buffer sends other groups to the fused kernel: other summation order)
        assert np.array_equal(g["acc_pot"][pact], acc_full[pact])                     # same groups, same lists, same sums
    s = bh.sync_status()
    assert s.sum_pc == int((t.gcount[sel] * st.npc[sel]).sum()) and s.sum_pp == int((t.gcount[sel] * st.npp[sel]).sum())


def test_call_order_and_arguments(BH):
    from paper_1106_1900_b200 import BhError
    pm, vel, prm = bh_inputs.make("c1", n=3000, seed=59)
    bh = BH(3000)
    bh.set_particles(pm, vel)
    with pytest.raises(BhError):
        bh.refresh_moments()                                    # no cells yet
    bh.tree_build(); bh.compute_forces(prm["theta"], prm["eps"])
    bh.kick_drift(0.01, 0.01)
    with pytest.raises(BhError):
        bh.compute_forces(prm["theta"], prm["eps"])             # moments are stale
    bh.refresh_moments()
    with pytest.raises(BhError):
        bh.compute_forces_active(prm["theta"], prm["eps"], torch.zeros(2999, dtype=torch.uint8, device="cuda"))
    with pytest.raises(BhError):
        bh.compute_forces_active(prm["theta"], prm["eps"], torch.zeros(3000, dtype=torch.uint8))
    bh.compute_forces_active(prm["theta"], prm["eps"], torch.zeros(3000, dtype=torch.uint8, device="cuda"))   # nobody active: a no-op walk
    s = bh.sync_status()
    assert s.sum_pc == 0 and s.sum_pp == 0
    bh.set_particles(pm, vel)
    with pytest.raises(BhError):
        bh.refresh_moments()                                    # new particles: the old cells do not describe them
