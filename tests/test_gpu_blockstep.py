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


# ------------------------------------------------------------------------------------------------ the scheme itself (A29)
def _block_pair(BH, n, seed, R, eta, dt_max=1.0 / 16, theta=0.6, eps=0.02, **cfg):
    """GPU context and oracle BlockState on the same particles, both initialised from the GPU's own fp32 forces."""
    pm, vel, _ = bh_inputs.make("c1", n=n, seed=seed)
    bh = BH(n, **cfg)
    g = gpu_tree(bh, pm, vel, theta, eps)
    bh.block_init(eps, eta, dt_max, R)
    st = oracle.tree_build(pm, vel)
    assert np.array_equal(st.pos, g["pos_mass"])
    st.accpot = g["acc_pot"].astype(np.float64)           # the held accelerations are the GPU's fp32 values on both sides
    bs = oracle.block_init(st, eps, eta, dt_max, R)
    return bh, bs, theta, eps


def _check_block_step(bh, bs, theta, eps, rebuild=False):
    """One block step on both sides.  The oracle replays it from the same state, takes its integer decisions from the same
    floats (the GPU's new accelerations), and everything but the forces must agree bit for bit."""
    bh.block_step(theta, eps, rebuild=rebuild)
    g = export_numpy(bh)
    b = bh.block_state()
    if rebuild:
        # the oracle: active set + predictor on the old order, then a fresh tree of the moved particles; its block state follows its own sort
        nxt, act = oracle.block_active(bs)
        oracle.lib().orc_block_predict(oracle.C.c_int64(bs.tree.n), oracle._p(bs.pos), oracle._p(bs.vel), oracle._p(bs.accb), oracle._p(act),
                                       oracle._p(bs.rung), oracle.C.c_float(bs.dt_max))
        st = oracle.tree_build(bs.pos, bs.vel, bs.ids)
        p = st.perm
        bs.pos, bs.vel, bs.ids, bs.tree = st.pos, st.vel, st.ids, st.tree
        bs.accb, bs.tick, bs.rung = bs.accb[p].copy(), bs.tick[p].copy(), bs.rung[p].copy()
        act = act[p].copy()
        assert np.array_equal(g["pos_mass"], bs.pos) and np.array_equal(g["id"].view(np.uint32), bs.ids)
        t = bs.tree
        sel = np.nonzero(np.add.reduceat(act.astype(np.int64), t.gbegin) > 0)[0].astype(np.int64)
        r = oracle.walk_forces(t, bs.pos, theta, eps, sel=sel)
        bs.npc, bs.npp, bs.acc_eval = r["npc"], r["npp"], r["accpot"]
        oracle.lib().orc_block_correct(oracle.C.c_int64(t.n), oracle._p(bs.vel), oracle._p(bs.accb), oracle._p(np.ascontiguousarray(g["acc_pot"])),
                                       oracle._p(act), oracle._p(bs.rung), oracle.C.c_float(bs.dt_max), oracle.C.c_uint32(nxt), oracle._p(bs.tick))
        oracle.rungs(bs.accb, act, bs.len_scale, bs.eta, bs.dt_max, bs.R, nxt, out=bs.rung)
        bs.now, bs.active = nxt, act
    else:
        bs = oracle.block_step(bs, theta, eps, acc_new=g["acc_pot"])
    t = bs.tree
    assert int(b["stats"].now_tick) == bs.now and int(b["stats"].n_active) == int(bs.active.sum())
    assert np.array_equal(b["active"], bs.active)
    assert np.array_equal(g["pos_mass"], bs.pos)                                  # predictor: bit-exact
    assert np.array_equal(g["cell_mom64"], t.mom64) and np.array_equal(g["cell_box"], t.box)   # partial refresh == full recomputation
    sel = np.nonzero(np.add.reduceat(bs.active.astype(np.int64), t.gbegin) > 0)[0]
    st = oracle.State(bs.pos, bs.vel, bs.ids, None, None, None, 0, t, bs.npc, bs.npp, bs.acc_eval)
    bad = compare_counts(g, st, sel=sel)
    assert not bad, "\n".join(bad)
    check_forces(g, st, sel=sel)
    assert np.array_equal(g["vel"], bs.vel)                                       # corrector with the same new accelerations: bit-exact
    assert np.array_equal(b["acc_held"], bs.accb) and np.array_equal(b["tick"], bs.tick) and np.array_equal(b["rung"], bs.rung)
    return bs, b


@pytest.mark.parametrize("n,R,eta,cfg", [(20000, 4, 0.2, {}), (4097, 3, 0.1, {}), (6000, 2, 0.3, dict(walk_mode=1)), (12000, 5, 0.15, dict(front_mode=1))])
def test_block_steps_track_the_oracle(BH, n, R, eta, cfg):
    bh, bs, theta, eps = _block_pair(BH, n, 83, R, eta, **cfg)
    b0 = bh.block_state()
    assert np.array_equal(b0["rung"], bs.rung) and len(set(bs.rung)) >= 2 and np.all(b0["tick"] == 0)
    fractions = []
    for step in range(6):
        bs, b = _check_block_step(bh, bs, theta, eps)
        fractions.append(int(b["stats"].n_active) / n)
    assert min(fractions) < 0.8                                                   # steps move a subset only (L264)
    assert b["stats"].interactions_now >= b["stats"].interactions_first > 0      # the cells only grow between rebuilds (L266)


def test_block_step_with_a_rebuild(BH):
    bh, bs, theta, eps = _block_pair(BH, 15000, 89, 3, 0.2)
    for step in range(5):
        bs, b = _check_block_step(bh, bs, theta, eps, rebuild=(step == 2))
        assert int(b["stats"].steps_since_rebuild) == (step + 1 if step < 2 else step - 1)
    assert b["stats"].interactions_first > 0


def test_block_scheme_reaches_the_macro_step_and_conserves_energy(BH):
    pm, vel, _ = bh_inputs.make("c1", n=8192, seed=97)
    theta, eps, R = 0.4, 0.05, 3
    bh = BH(8192)
    g0 = gpu_tree(bh, pm, vel, theta, eps)
    bh.block_init(eps, 0.1, 1.0 / 16, R)

    def energy(g):
        d = oracle.direct(g["pos_mass"], eps)
        m = g["pos_mass"][:, 3].astype(np.float64)
        return 0.5 * np.sum(m * np.sum(g["vel"][:, :3].astype(np.float64) ** 2, axis=1)) + 0.5 * np.sum(m * d[:, 3])

    e0 = energy(g0)
    steps = 0
    while True:
        bh.block_step(theta, eps)
        steps += 1
        if int(bh.block_state(arrays=False)["stats"].now_tick) >= 1 << R:
            break
    b = bh.block_state()
    assert np.all(b["tick"] == 1 << R) and 2 <= steps <= 1 << R                 # everybody is synchronised at the end of the longest step
    assert abs((energy(export_numpy(bh)) - e0) / e0) < 2e-4


def test_block_call_order(BH):
    from paper_1106_1900_b200 import BhError
    pm, vel, prm = bh_inputs.make("c1", n=3000, seed=101)
    bh = BH(3000)
    bh.set_particles(pm, vel)
    bh.tree_build()
    with pytest.raises(BhError):
        bh.block_init(0.01, 0.2, 1 / 16, 3)                 # no forces yet
    with pytest.raises(BhError):
        bh.block_step(0.5, 0.01)                            # not initialised
    bh.compute_forces(0.5, 0.01)
    for bad in ((0.0, 0.2, 1 / 16, 3), (0.01, 0.0, 1 / 16, 3), (0.01, 0.2, 0.0, 3), (0.01, 0.2, 1 / 16, 21)):
        with pytest.raises(BhError):
            bh.block_init(*bad)
    bh.block_init(0.01, 0.2, 1 / 16, 3)
    bh.block_step(0.5, 0.01)
    bh.set_particles(pm, vel)
    with pytest.raises(BhError):
        bh.block_step(0.5, 0.01)                            # new particles: the block state is gone


def test_active_walk_is_bit_identical_with_shared_super_group_walks(BH):
    """At this size the list walk shares the common part of the walks of neighbouring groups (walk_lists.cu); which groups
    share must depend on the group index only, so a walk of an active subset reproduces the full walk's sums bit for bit,
    and the counts stay those of the oracle."""
    n = 400000
    pm, vel, prm = bh_inputs.make("c2", n=n, seed=103)
    bh = BH(n)
    g = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
    assert g["stats"].sum_mac < 1100 * g["n_groups"]                 # the shared walk is in use: far fewer MAC tests than ~1300 per group
    acc_full = g["acc_pot"].copy()
    rng = np.random.default_rng(7)
    active = (rng.random(n) < 0.03).astype(np.uint8)
    bh.kick_drift(0.0, 0.0); bh.refresh_moments()
    bh.compute_forces_active(prm["theta"], prm["eps"], torch.from_numpy(active).cuda())
    g2 = export_numpy(bh)
    gb = g2["group_begin"].astype(np.int64)
    gact = np.add.reduceat(active.astype(np.int64), gb[:-1]) > 0
    walked = np.repeat(gact, np.diff(gb))
    assert 0.2 < gact.mean() < 0.9
    assert np.array_equal(g2["acc_pot"][walked], acc_full[walked]) and np.array_equal(g2["acc_pot"][~walked], acc_full[~walked])
    assert np.array_equal(g2["group_npc"][gact], g["group_npc"][gact]) and np.all(g2["group_npc"][~gact] == 0)
    # counts against the oracle on a sample of the walked groups
    st = oracle.tree_build(pm, vel)
    sel = np.nonzero(gact)[0][::40].astype(np.int64)
    oracle.compute_forces(st, prm["theta"], prm["eps"], sel=sel)
    bad = compare_counts(g2, st, sel=sel)
    assert not bad, "\n".join(bad)
    check_forces(g2, st, sel=sel)
    # and a context that walks every group on its own gives the same counts (the order of the entries, hence the last bits, differ)
    priv = BH(n, walk_private=1)
    g3 = gpu_tree(priv, pm, vel, prm["theta"], prm["eps"])
    assert np.array_equal(g3["group_npc"], g["group_npc"]) and np.array_equal(g3["group_npp"], g["group_npp"])
    assert g3["stats"].sum_mac > 1200 * g3["n_groups"]
    err = np.abs(g3["acc_pot"][:, :3] - acc_full[:, :3]).max() / np.abs(acc_full[:, :3]).max()
    assert err < 1e-5
