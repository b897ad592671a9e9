"""GPU parity tests: the CUDA path, called through the C ABI, against the CPU oracle on the same seeded inputs.

Sizes the oracle finishes in seconds, spanning several tiles (sort tile 4096, tree tile 256, scan tile 2048) and
ragged tails, plus the degenerate cases (one particle, a root leaf, coincident particles -> level-20 overflow leaf).
"""
import numpy as np
import pytest
import torch

import bh_inputs
import oracle
from parity_common import (check_forces, compare_counts, compare_tree, export_numpy, force_errors, gpu_tree,
                           oracle_state)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def BH():
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import BarnesHut
    return BarnesHut


def _full_parity(BH, pm, vel, theta, eps, mac=0, **cfg):
    bh = BH(pm.shape[0], **cfg)
    g = gpu_tree(bh, pm, vel, theta, eps, mac=mac)
    st = oracle_state(pm, vel, theta, eps, nleaf=cfg.get("nleaf", 0) or 16, ncrit=cfg.get("ncrit", 0) or 64, mac=mac)
    bad = compare_tree(g, st)
    compare_counts(g, st, problems=bad)
    assert not bad, "\n".join(bad)
    e = check_forces(g, st)
    bh.close()
    return g, st, e


@pytest.mark.parametrize("front_mode", [0, 1, 2])
@pytest.mark.parametrize("cfg,n", [("c1", 16384), ("c1", 5000), ("c1", 4097), ("c1", 257), ("c3", 30000), ("c3", 12289)])
def test_full_pipeline_parity(BH, cfg, n, front_mode):
    """Through every front end: the one-launch front end with the short sort (leading key bits + fix-up), the one launch per
    pass of large inputs, and the one-launch front end with all 8 passes."""
    pm, vel, prm = bh_inputs.make(cfg, n=n)
    g, _, _ = _full_parity(BH, pm, vel, prm["theta"], prm["eps"], front_mode=front_mode)
    assert g["stats"].sort_retries == 0


def _with_clump(n, clump, radius, seed):
    """A c1 sphere with `clump` of its particles moved into a ball of `radius` around one of them (radius 0: coincident)."""
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=seed)
    rng = np.random.Generator(np.random.Philox(seed + 1))
    idx = rng.choice(n, size=clump, replace=False)
    centre = pm[idx[0], :3].astype(np.float64)
    off = rng.standard_normal((clump, 3)) * radius
    pm[idx, :3] = (centre + off).astype(np.float32)
    return pm, vel, prm


@pytest.mark.parametrize("front_mode", [0, 1])
@pytest.mark.parametrize("n,clump,radius,retries", [(20000, 48, 3e-4, 0), (20000, 30, 0.0, 0), (20000, 700, 3e-4, 1), (9000, 300, 0.0, 1), (4097, 4000, 1e-4, 1)])
def test_short_sort_on_clustered_keys(BH, n, clump, radius, retries, front_mode):
    """Runs of keys that agree on the leading bits the short sort looks at: a short run is finished by the fix-up (order of the
    trailing bits, equal keys in their original order), a long one makes the device redo the sort in full.  The permutation is
    bit-exact either way."""
    pm, vel, prm = _with_clump(n, clump, radius, seed=300 + clump)
    bh = BH(n, front_mode=front_mode)
    g = gpu_tree(bh, pm, vel, prm["theta"], 0.05)
    st = oracle_state(pm, vel, prm["theta"], 0.05)
    # the input really has what the case is about: the longest run of equal leading 40 bits
    top = st.keys >> np.uint64(20)
    runs = np.diff(np.flatnonzero(np.concatenate([[True], top[1:] != top[:-1], [True]])))
    assert (runs.max() > 128) == bool(retries) and runs.max() > 16
    bad = compare_tree(g, st)
    compare_counts(g, st, problems=bad)
    assert not bad, "\n".join(bad)
    if front_mode == 0:
        assert g["stats"].sort_retries == retries
    # a second build on the same context (the retry flag and the barrier words are back to their idle values)
    bh.set_particles(pm, vel)
    bh.tree_build()
    bh.compute_forces(prm["theta"], 0.05)
    g2 = export_numpy(bh)
    assert np.array_equal(g2["perm"], g["perm"]) and np.array_equal(g2["key"], g["key"])
    if front_mode == 0:
        assert g2["stats"].sort_retries == 2 * retries
    bh.close()


def _many_clumps(n, clumps, size, radius, seed):
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=seed)
    rng = np.random.Generator(np.random.Philox(seed + 1))
    idx = rng.choice(n, size=clumps * size, replace=False).reshape(clumps, size)
    for row in idx:
        centre = pm[row[0], :3].astype(np.float64)
        pm[row, :3] = (centre + rng.standard_normal((size, 3)) * radius).astype(np.float32)
    return pm, vel, prm


@pytest.mark.parametrize("seed,size", [(611, 100), (612, 100), (621, 60), (622, 60), (623, 60)])
def test_short_sort_runs_across_tile_boundaries(BH, seed, size):
    """Runs of ~100 / ~60 keys with equal leading bits, many of them, so that some lie across the boundary between two sort tiles:
    inside the halo of 64 the fix-up finishes them from either side; a run that reaches further into the neighbouring tile
    must be given up (full re-sort).  What the device has to decide is predicted here from the oracle's keys and the tiling."""
    import torch
    n = 30000
    pm, vel, prm = _many_clumps(n, 6000 // size, size, 2e-4, seed)
    st = oracle_state(pm, vel, prm["theta"], 0.05)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    tile = min(max(-(-(-(-n // sms)) // 1024) * 1024, 1024), 8192)
    top = st.keys >> np.uint64(20)
    edges = np.flatnonzero(np.concatenate([[True], top[1:] != top[:-1], [True]]))
    halo, giveup, crossing = 64, False, 0
    for a, b in zip(edges[:-1], edges[1:]):
        if b - a > 2 * halo:
            giveup = True
        for w0 in range(tile, n, tile):
            if a < w0 < b:
                crossing += 1
                if w0 - a >= halo or b - w0 >= halo:      # the window of one of the two tiles ends inside the run
                    giveup = True
    assert crossing > 0 and giveup == (size > 64)
    bh = BH(n)
    g = gpu_tree(bh, pm, vel, prm["theta"], 0.05)
    bad = compare_tree(g, st)
    compare_counts(g, st, problems=bad)
    assert not bad, "\n".join(bad)
    assert g["stats"].sort_retries == (1 if giveup else 0), (giveup, crossing)
    bh.close()


@pytest.mark.parametrize("cfg,n", [("c1", 20000), ("c3", 12289)])
def test_short_sort_of_large_inputs_follows_the_previous_tree(BH, cfg, n):
    """The one-launch-per-pass front end (any n): the first build sorts in full; the next one sorts only the leading 3 x levels
    bits of the previous tree (whole digits) and finishes the rest in the fix-up; a particle set that is far more clustered
    than the previous tree suggests makes the device sort again in full.  Bit-exact against the oracle every time."""
    pm, vel, prm = bh_inputs.make(cfg, n=n, seed=77)
    bh = BH(n, front_mode=1)
    g = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
    assert g["stats"].sort_passes == 8 and g["stats"].sort_retries == 0
    levels = g["stats"].n_levels
    st = oracle_state(pm, vel, prm["theta"], prm["eps"])
    g2 = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
    assert g2["stats"].sort_passes == min(8, -(-3 * levels // 8)) < 8 and g2["stats"].sort_retries == 0
    bad = compare_tree(g2, st)
    compare_counts(g2, st, problems=bad)
    assert not bad, "\n".join(bad)
    if cfg == "c1":
        # equal keys inside a run the fix-up finishes (40 coincident particles, the shallow tree's hint): their original order stays
        pm5, vel5, _ = _with_clump(n, 40, 0.0, seed=79)
        g5 = gpu_tree(bh, pm5, vel5, prm["theta"], 0.05)
        assert g5["stats"].sort_passes < 8 and g5["stats"].sort_retries == 0
        st5 = oracle_state(pm5, vel5, prm["theta"], 0.05)
        assert np.unique(st5.keys).size < n
        bad = compare_tree(g5, st5)
        assert not bad, "\n".join(bad)
        g = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])         # back to the plain set (and a shallow tree for the next hint)
        g = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
    pm3, vel3, _ = _with_clump(n, 900, 3e-4, seed=78) if cfg == "c1" else (None, None, None)
    if pm3 is not None:
        g3 = gpu_tree(bh, pm3, vel3, prm["theta"], 0.05)
        assert g3["stats"].sort_passes < 8 and g3["stats"].sort_retries == 1
        st3 = oracle_state(pm3, vel3, prm["theta"], 0.05)
        bad = compare_tree(g3, st3)
        compare_counts(g3, st3, problems=bad)
        assert not bad, "\n".join(bad)
        g4 = gpu_tree(bh, pm3, vel3, prm["theta"], 0.05)          # the deep tree of the clump now says how much to sort
        assert g4["stats"].sort_retries == 1 and np.array_equal(g4["perm"], g3["perm"])
    bh.close()


@pytest.mark.parametrize("theta,eps", [(0.5, 0.01), (0.3, 0.0), (1.0, 0.05)])
def test_parity_other_opening_angles_and_softening(BH, theta, eps):
    pm, vel, _ = bh_inputs.make("c1", n=8192, seed=7)
    _full_parity(BH, pm, vel, theta, eps)


@pytest.mark.parametrize("cfg", [dict(walk_mode=1), dict(list_entries=3000), dict(list_entries=40000), dict(list_entries=1)])
def test_walk_paths_agree(BH, cfg):
    """Fused kernel only; list buffer too small for most / some / all groups (deferred to the fused kernel): same counts, same forces."""
    pm, vel, prm = bh_inputs.make("c1", n=6000, seed=13)
    _full_parity(BH, pm, vel, prm["theta"], prm["eps"], **cfg)


@pytest.mark.parametrize("cfg", [dict(list_entries=1 << 20), dict(walk_waves=5), dict(walk_waves=2, list_entries=1 << 22)])
def test_walk_in_several_waves(BH, cfg):
    """Several waves (forced by a small list buffer, or asked for): the list walk of wave w + 1 runs beside the evaluation of
    wave w on internal streams; same counts, same forces."""
    pm, vel, prm = bh_inputs.make("c1", n=40000, seed=17)
    _full_parity(BH, pm, vel, prm["theta"], prm["eps"], **cfg)


@pytest.mark.parametrize("cfg,n,theta,extra", [("c1", 16384, 0.75, {}), ("c1", 4097, 0.5, {}), ("c3", 12289, 0.6, {}), ("c1", 6000, 0.75, dict(walk_mode=1)),
                                               ("c1", 6000, 0.75, dict(list_entries=40000)), ("c1", 40000, 0.75, dict(walk_waves=3))])
def test_minimum_distance_mac_parity(BH, cfg, n, theta, extra):
    """The minimum-distance MAC (A28) through every walk path: counts bit-exact, forces within tolerance."""
    pm, vel, prm = bh_inputs.make(cfg, n=n, seed=41)
    g, st, _ = _full_parity(BH, pm, vel, theta, prm["eps"], mac=1, **extra)
    # and it is a different walk from Eq.1's: more interactions on the same tree
    st0 = oracle_state(pm, vel, theta, prm["eps"], forces=False)
    assert g["group_npc"].sum() + g["group_npp"].sum() > st0.npc.sum() + st0.npp.sum()


def test_switching_the_mac_needs_no_rebuild(BH):
    pm, vel, prm = bh_inputs.make("c1", n=5000, seed=43)
    bh = BH(5000)
    g0 = gpu_tree(bh, pm, vel, 0.75, prm["eps"])
    bh.set_mac(1)
    with pytest.raises(Exception):
        bh.leapfrog_step(0.75, prm["eps"], prm["dt"])          # forces of the old criterion are no longer valid
    bh.compute_forces(0.75, prm["eps"])
    g1 = export_numpy(bh)
    st1 = oracle_state(pm, vel, 0.75, prm["eps"], mac=1)
    bad = compare_counts(g1, st1)
    assert not bad, "\n".join(bad)
    check_forces(g1, st1)
    bh.set_mac(0)
    bh.compute_forces(0.75, prm["eps"])
    g2 = export_numpy(bh)
    assert np.array_equal(g2["group_npc"], g0["group_npc"]) and np.array_equal(g2["acc_pot"], g0["acc_pot"])
    with pytest.raises(Exception):
        bh.set_mac(2)


@pytest.mark.parametrize("n", [1, 2, 16, 17, 64, 65])
def test_tiny_inputs(BH, n):
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=11)
    bh = BH(max(n, 1))
    g = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
    st = oracle_state(pm, vel, prm["theta"], prm["eps"])
    bad = compare_tree(g, st)
    compare_counts(g, st, problems=bad)
    assert not bad, "\n".join(bad)
    if n > 1:
        check_forces(g, st)
    else:
        assert np.all(g["acc_pot"] == 0.0)


def test_other_leaf_and_group_sizes(BH):
    pm, vel, prm = bh_inputs.make("c1", n=6000, seed=3)
    _full_parity(BH, pm, vel, prm["theta"], prm["eps"], nleaf=8, ncrit=32)
    _full_parity(BH, pm, vel, prm["theta"], prm["eps"], nleaf=32, ncrit=16)


def test_coincident_particles_overflow_leaf(BH):
    # 150 particles at one point (level-20 overflow leaf, chunked groups) inside a small Plummer sphere
    pm, vel, prm = bh_inputs.make("c1", n=2000, seed=5)
    pm[100:250, :3] = pm[100, :3]
    g, st, e = _full_parity(BH, pm, vel, prm["theta"], 0.05)
    assert g["stats"].n_levels == 21
    assert st.tree.pcount[st.tree.level == 20].max() == 150


def test_nonfinite_input_is_reported(BH):
    from paper_1106_1900_b200 import BhError
    pm, vel, prm = bh_inputs.make("c1", n=3000)
    for bad in (np.nan, np.inf):
        q = pm.copy(); q[1234, 2] = bad
        bh = BH(3000)
        bh.set_particles(q, vel)
        bh.tree_build()
        assert bh.sync_status(check=False).status == -5
    q = pm.copy(); q[17, 3] = 0.0
    bh = BH(3000)
    bh.set_particles(q, vel)
    bh.tree_build()
    with pytest.raises(BhError):
        bh.sync_status()


def test_call_order_and_arguments_are_checked(BH):
    from paper_1106_1900_b200 import BhError
    pm, vel, prm = bh_inputs.make("c1", n=1000)
    bh = BH(1000)
    with pytest.raises(BhError):
        bh.tree_build()                     # no particles yet
    bh.set_particles(pm, vel)
    with pytest.raises(BhError):
        bh.compute_forces(0.5, 0.01)        # no tree yet
    bh.tree_build()
    with pytest.raises(BhError):
        bh.leapfrog_step(0.5, 0.01, 0.01)   # no forces yet
    for theta, eps in ((0.0, 0.01), (-1.0, 0.01), (float("nan"), 0.01), (0.5, -0.1)):
        with pytest.raises(BhError):
            bh.compute_forces(theta, eps)
    with pytest.raises(BhError):
        bh.set_particles(np.zeros((1001, 4), np.float32))   # n > n_max
    # a too-small cell capacity is a deferred device error, not a crash
    small = BH(1000, max_cells=10)
    small.set_particles(pm, vel)
    small.tree_build()
    assert small.sync_status(check=False).status == -6


def test_device_and_pinned_inputs_and_ids(BH):
    pm, vel, prm = bh_inputs.make("c1", n=5000, seed=9)
    ids = (np.arange(5000, dtype=np.uint32)[::-1] * 3 + 1).copy()
    st = oracle_state(pm, vel, prm["theta"], prm["eps"], ids=ids)
    for conv in (lambda a: torch.from_numpy(a).cuda(), lambda a: torch.from_numpy(a).pin_memory()):
        bh = BH(5000)
        keep = (conv(pm), conv(vel), conv(ids.view(np.int32)))
        bh.set_particles(*keep)
        bh.tree_build()
        bh.compute_forces(prm["theta"], prm["eps"])
        g = export_numpy(bh)
        assert np.array_equal(g["id"].view(np.uint32), st.ids)
        assert not compare_tree(g, st)
        out = np.empty((5000, 4), np.float32)
        bh.get_particles(acc_pot=out)
        torch.cuda.synchronize()
        assert np.array_equal(out, g["acc_pot"])


def test_leapfrog_steps_track_the_oracle(BH):
    """Per-call parity: after each GPU step the oracle repeats that step from the GPU's state."""
    pm, vel, prm = bh_inputs.make("c1")
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    bh = BH(pm.shape[0])
    g = gpu_tree(bh, pm, vel, theta, eps)
    for step in range(2):
        # the oracle starts from the GPU's synchronised state (sorted order, ids, fp32 accelerations)
        st = oracle.tree_build(g["pos_mass"].copy(), g["vel"].copy(), g["id"].view(np.uint32).copy())
        st.accpot = g["acc_pot"].astype(np.float64)
        assert np.array_equal(st.perm, np.arange(st.tree.n, dtype=np.uint32))   # already sorted
        st2 = oracle.leapfrog_step(st, theta, eps, dt)
        bh.leapfrog_step(theta, eps, dt)
        g = export_numpy(bh)
        # positions after the drift, keys, tree, moments: bit-exact.  Velocities carry the closing kick with the NEW
        # accelerations, which agree only to the force tolerance, so they are compared below with a bound instead.
        bad = compare_tree(g, st2, check_vel=False)
        compare_counts(g, st2, problems=bad)
        assert not bad, f"step {step}:\n" + "\n".join(bad)
        check_forces(g, st2)
        # velocities after the closing kick: same fp32 fma on accelerations that differ by <= 1e-4 relative
        dv = np.abs(g["vel"][:, :3] - st2.vel[:, :3]).max()
        assert dv < 1e-5, dv


def test_energy_and_momentum_over_steps(BH):
    pm, vel, prm = bh_inputs.make("c1")
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    bh = BH(pm.shape[0])
    g = gpu_tree(bh, pm, vel, theta, eps)

    def energy(g):
        m = g["pos_mass"][:, 3].astype(np.float64)
        return 0.5 * np.sum(m * np.sum(g["vel"][:, :3].astype(np.float64) ** 2, axis=1)) + 0.5 * np.sum(m * g["acc_pot"][:, 3])

    e0 = energy(g)
    for _ in range(8):
        bh.leapfrog_step(theta, eps, dt)
    g = export_numpy(bh)
    assert abs((energy(g) - e0) / e0) < 2e-4
    m = g["pos_mass"][:, 3].astype(np.float64)
    a = g["acc_pot"][:, :3].astype(np.float64)
    assert np.linalg.norm((m[:, None] * a).sum(0)) / np.sum(m * np.linalg.norm(a, axis=1)) < 5e-4
    assert sorted(g["id"].view(np.uint32)) == list(range(pm.shape[0]))


def test_deterministic(BH):
    pm, vel, prm = bh_inputs.make("c1", n=10000)
    runs = []
    for _ in range(2):
        bh = BH(10000)
        g = gpu_tree(bh, pm, vel, prm["theta"], prm["eps"])
        runs.append({k: np.array(v, copy=True) for k, v in g.items() if isinstance(v, np.ndarray)})
    for k in runs[0]:
        if k == "acc_pot":      # fp32 sums: order inside a group is fixed, so these are reproducible too
            assert np.array_equal(runs[0][k], runs[1][k]), k
        else:
            assert np.array_equal(runs[0][k], runs[1][k]), k


def test_theta_to_zero_is_the_direct_sum(BH):
    pm, vel, _ = bh_inputs.make("c1", n=1500)
    bh = BH(1500)
    g = gpu_tree(bh, pm, vel, 1e-6, 0.01)
    ps = oracle.tree_build(pm, vel).pos                     # the oracle's own sorted particles ...
    assert np.array_equal(g["pos_mass"], ps)                # ... which are the GPU's, bit for bit
    d = oracle.direct(ps, 0.01)
    a = g["acc_pot"].astype(np.float64)
    err = np.linalg.norm(a[:, :3] - d[:, :3], axis=1) / np.linalg.norm(d[:, :3], axis=1)
    assert np.sqrt(np.mean(err ** 2)) < 1e-5 and err.max() < 1e-4
    assert np.all(g["group_npc"] + g["group_npp"] == 1500)


def test_stage_timing_and_walk_timeline(BH):
    """The profiling aids of the boundary: per-stage CUDA-event times and the device timeline of the walk."""
    pm, vel, prm = bh_inputs.make("c1", n=40000, seed=73)
    for waves in (0, 3):
        bh = BH(40000, walk_waves=waves)
        bh.set_particles(pm, vel)
        bh.set_stage_timing(True)
        bh.tree_build()
        bh.compute_forces(prm["theta"], prm["eps"])
        ms = bh.stage_ms()
        assert set(ms) == {"bbox", "keys", "sort", "reorder", "cells", "groups", "moments", "record", "walk", "lists", "eval"}
        assert all(v >= 0.0 for v in ms.values()) and ms["walk"] > 0.0 and ms["sort"] > 0.0
        tl = bh.walk_timeline()
        if waves == 0:
            assert ms["lists"] > 0.0 and ms["eval"] > 0.0 and ms["lists"] + ms["eval"] <= ms["walk"] * 1.001
            assert len(tl) == 1
        else:
            assert ms["lists"] == 0.0 and ms["eval"] == 0.0          # the kernels of a pipelined walk overlap: no split
            assert len(tl) == 3
        for ls, le, es, ee in tl:
            assert 0 <= ls <= le and es <= ee and le <= ee           # a wave is evaluated after it has been listed
        bh.close()
