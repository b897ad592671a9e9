"""bh_bind_particles / bh_land_particles (the particles stay on the GPU): the
caller's own device arrays are the simulation state.  The steps are replayed by the oracle from the GPU's state (positions
and ids bit for bit, counts bit for bit, forces in tolerance), the run is bit-identical to one that copied the same
particles in with bh_set_particles, and the pointers bh_export_tree reports ARE the caller's tensors -- there is no copy to
hide.  The caller's arrays sit between guard rows that must come through untouched."""
import ctypes as C

import numpy as np
import pytest
import torch

import bh_inputs
import oracle
from parity_common import check_forces, compare_counts, compare_tree, export_numpy, gpu_tree

pytestmark = pytest.mark.gpu

GUARD = 64          # rows of sentinel before and after every array


@pytest.fixture(scope="module")
def BH():
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import BarnesHut
    return BarnesHut


def export_both(b):
    """One bh_export_tree: the torch views (for their pointers) and the same arrays as numpy."""
    t = b.export_tree()
    g = {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in t.items()}
    g["key"] = g["key"].astype(np.uint64)
    g["cell_prefix"] = g["cell_prefix"].astype(np.uint64)
    return t, g


class CallerArrays:
    """pos, vel, acc (float32[n,4]) and id (int32[n]) carved out of larger tensors full of a sentinel."""

    def __init__(self, pm, vel):
        n = pm.shape[0]
        self.n = n
        self.raw = [torch.full((n + 2 * GUARD, 4), -7.25, dtype=torch.float32, device="cuda") for _ in range(3)]
        self.raw_id = torch.full((n + 2 * GUARD,), -77, dtype=torch.int32, device="cuda")
        self.pos, self.vel, self.acc = (r[GUARD: GUARD + n] for r in self.raw)
        self.ids = self.raw_id[GUARD: GUARD + n]
        self.pos.copy_(torch.from_numpy(pm))
        self.vel.copy_(torch.from_numpy(vel))
        self.ids.copy_(torch.arange(n, dtype=torch.int32))
        torch.cuda.synchronize()

    def guards_intact(self):
        ok = all(bool((r[:GUARD] == -7.25).all()) and bool((r[GUARD + self.n:] == -7.25).all()) for r in self.raw)
        return ok and bool((self.raw_id[:GUARD] == -77).all()) and bool((self.raw_id[GUARD + self.n:] == -77).all())


@pytest.mark.parametrize("n,front_mode", [(16384, 0), (20001, 1), (300_000, 0)])
def test_bound_arrays_are_the_state(BH, n, front_mode):
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=307)
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    ca = CallerArrays(pm, vel)
    bh = BH(n, front_mode=front_mode)
    bh.bind_particles(ca.pos, ca.vel, ca.acc, ca.ids)
    ref = BH(n, front_mode=front_mode)                    # the same run with the particles copied in
    ref.set_particles(pm, vel)
    for b in (bh, ref):
        b.tree_build(); b.compute_forces(theta, eps)
    (t, g), _ = export_both(bh), export_both(ref)
    assert t["acc_pot"].data_ptr() == ca.acc.data_ptr()                      # forces land in the caller's array, always
    assert t["pos_mass"].data_ptr() != ca.pos.data_ptr()                     # one build: the sorted particles are in the workspace
    st = oracle.compute_forces(oracle.tree_build(pm, vel), theta, eps)
    bad = compare_tree(g, st)
    compare_counts(g, st, problems=bad)
    assert not bad, "\n".join(bad)
    check_forces(g, st)
    for step in range(1, 5):
        st = oracle.tree_build(g["pos_mass"].copy(), g["vel"].copy(), g["id"].view(np.uint32).copy())
        st.accpot = g["acc_pot"].astype(np.float64)
        st2 = oracle.leapfrog_step(st, theta, eps, dt)
        bh.leapfrog_step(theta, eps, dt); ref.leapfrog_step(theta, eps, dt)
        (t, g), (_, gr) = export_both(bh), export_both(ref)
        in_callers = step % 2 == 1                                           # builds since the binding: step + 1
        assert (t["pos_mass"].data_ptr() == ca.pos.data_ptr()) == in_callers
        assert (t["vel"].data_ptr() == ca.vel.data_ptr()) == in_callers and (t["id"].data_ptr() == ca.ids.data_ptr()) == in_callers
        assert t["acc_pot"].data_ptr() == ca.acc.data_ptr()
        bad = compare_tree(g, st2, check_vel=False)
        compare_counts(g, st2, problems=bad)
        assert not bad, f"step {step}:\n" + "\n".join(bad)
        check_forces(g, st2)
        for k in ("pos_mass", "vel", "acc_pot", "id", "key", "group_npc", "group_npp"):
            assert np.array_equal(g[k], gr[k]), (step, k)
        if in_callers:                                                       # the caller reads its own tensors, no call needed
            assert np.array_equal(ca.pos.cpu().numpy(), st2.pos) and np.array_equal(ca.ids.cpu().numpy().view(np.uint32), st2.ids)
            assert np.array_equal(ca.vel.cpu().numpy(), g["vel"]) and np.array_equal(ca.acc.cpu().numpy(), g["acc_pot"])
    # exactly the kernels of the copied-in run and nothing else -- no copy kernel stands in for the missing memcpy.  (The
    # copied-in run has more: the iota that numbers its ids and, with the one-launch front end, the first build's reorder
    # as a launch of its own, because its velocities were still arriving when that build was enqueued.)
    assert ref.sync_status().launches - bh.sync_status().launches == (2 if front_mode == 0 else 1)
    assert ca.guards_intact()


def test_landing_after_an_odd_number_of_builds(BH):
    n = 20000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=311)
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    ca = CallerArrays(pm, vel)
    bh = BH(n)
    bh.bind_particles(ca.pos, ca.vel, ca.acc, ca.ids)
    bh.tree_build(); bh.compute_forces(theta, eps)
    bh.leapfrog_step(theta, eps, dt); bh.leapfrog_step(theta, eps, dt)       # three builds: the state is in the workspace
    g = export_numpy(bh)
    assert not np.array_equal(ca.pos.cpu().numpy(), g["pos_mass"])
    launches = bh.sync_status().launches
    bh.land_particles()
    t = bh.export_tree()
    assert t["pos_mass"].data_ptr() == ca.pos.data_ptr() and t["id"].data_ptr() == ca.ids.data_ptr()
    for mine, k in ((ca.pos, "pos_mass"), (ca.vel, "vel"), (ca.acc, "acc_pot")):
        assert np.array_equal(mine.cpu().numpy(), g[k]), k
    assert np.array_equal(ca.ids.cpu().numpy(), g["id"])
    bh.land_particles()                                                      # already there: nothing happens
    assert bh.sync_status().launches == launches + 1                         # (+ 1: the export kernel of export_tree above)
    # tree and forces are still valid: the next step continues the run of a context that never landed
    ref = BH(n)
    gpu_tree(ref, pm, vel, theta, eps)
    for _ in range(3):
        ref.leapfrog_step(theta, eps, dt)
    bh.leapfrog_step(theta, eps, dt)
    g, gr = export_numpy(bh), export_numpy(ref)
    for k in ("pos_mass", "vel", "acc_pot", "id", "group_npc", "group_npp"):
        assert np.array_equal(g[k], gr[k]), k
    assert ca.guards_intact()


def test_bound_arrays_through_the_step_graph_and_back_to_the_workspace(BH):
    n = 20000
    pm, vel, prm = bh_inputs.make("c1", n=n, seed=313)
    theta, eps, dt = prm["theta"], prm["eps"], prm["dt"]
    ca = CallerArrays(pm, vel)
    bh, ref = BH(n), BH(n)
    bh.bind_particles(ca.pos, ca.vel, ca.acc, ca.ids)
    bh.tree_build(); bh.compute_forces(theta, eps)
    gpu_tree(ref, pm, vel, theta, eps)
    bh.step_graph_build(theta, eps, dt)
    for _ in range(3):
        bh.step_graph_launch(); ref.leapfrog_step(theta, eps, dt)
    g, gr = export_numpy(bh), export_numpy(ref)
    for k in ("pos_mass", "vel", "acc_pot", "id"):
        assert np.array_equal(g[k], gr[k]), k
    assert np.array_equal(ca.pos.cpu().numpy(), g["pos_mass"])               # four builds: the caller's arrays are current
    # bh_set_particles releases the caller's arrays: they are not written any more
    before = [x.clone() for x in (ca.pos, ca.vel, ca.acc)]
    bh.set_particles(pm, vel)
    bh.tree_build(); bh.compute_forces(theta, eps); bh.leapfrog_step(theta, eps, dt); bh.leapfrog_step(theta, eps, dt)
    torch.cuda.synchronize()
    for x, y in zip(before, (ca.pos, ca.vel, ca.acc)):
        assert torch.equal(x, y)
    t = bh.export_tree()
    assert t["acc_pot"].data_ptr() != ca.acc.data_ptr()
    assert ca.guards_intact()


def test_bind_arguments(BH):
    from paper_1106_1900_b200 import BhError, load_library
    n = 4096
    pm, vel, _ = bh_inputs.make("c1", n=n, seed=317)
    ca = CallerArrays(pm, vel)
    bh = BH(n)
    lib = load_library()
    p, v, a, i = (C.c_void_p(x.data_ptr()) for x in (ca.pos, ca.vel, ca.acc, ca.ids))
    assert lib.bh_bind_particles(bh.h, n + 1, p, v, a, i) == -1              # more than n_max
    assert lib.bh_bind_particles(bh.h, 0, p, v, a, i) == -1
    assert lib.bh_bind_particles(bh.h, n, None, v, a, i) == -1
    assert lib.bh_bind_particles(bh.h, n, C.c_void_p(ca.pos.data_ptr() + 4), v, a, i) == -1      # float4 rows must be 16-byte aligned
    assert lib.bh_bind_particles(bh.h, n, C.c_void_p(pm.ctypes.data), v, a, i) == -1             # host memory
    with pytest.raises(BhError):
        bh.bind_particles(ca.pos, ca.vel, ca.acc, ca.ids.to(torch.int64))
    with pytest.raises(BhError):
        bh.tree_build()                                                       # nothing bound yet
    assert lib.bh_land_particles(bh.h, None) == -3
    assert lib.bh_bind_particles(bh.h, n, p, v, a, i) == 0
    with pytest.raises(BhError):
        bh.compute_forces(0.7, 0.01)                                          # bound, but no tree yet
