"""Pins P6-P14 for the CPU oracle: moments, p-c formula, walk + forces, potential, leapfrog (no GPU).

The checks are closed forms, textbook limits, brute force and invariants -- none re-uses the
oracle's own formulas.
"""
import math

import numpy as np
import pytest

import bh_inputs
import oracle


def _state(cfg="c1", n=4096, seed=None):
    pm, v, prm = bh_inputs.make(cfg, n=n, seed=seed)
    return oracle.tree_build(pm, v), prm


def _relerr(a, ref):
    return np.linalg.norm(a[:, :3] - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)


# ---------------------------------------------------------------- P6: moments
def test_root_moments_match_direct_sums_and_boxes_tight():
    st, _ = _state("c1", 16384)
    t, p = st.tree, st.pos.astype(np.float64)
    m, x = p[:, 3], p[:, :3]
    M = m.sum()
    com = (m[:, None] * x).sum(0) / M
    r = x - com
    Q = np.einsum("i,ij,ik->jk", m, r, r)
    got = t.mom64[0]
    assert abs(got[0] - M) < 1e-13 * M
    assert np.allclose(got[1:4], com, rtol=0, atol=1e-12)
    want = np.array([Q[0, 0], Q[1, 1], Q[2, 2], Q[0, 1], Q[0, 2], Q[1, 2]])
    assert np.allclose(got[4:], want, rtol=1e-11, atol=1e-13)
    # every cell: box is the exact min / max of its particles; moments of leaves by direct sums
    for c in range(0, t.ncells, 37):
        s = slice(int(t.pbegin[c]), int(t.pbegin[c] + t.pcount[c]))
        assert np.array_equal(t.box[c, :3], st.pos[s, :3].min(0)) and np.array_equal(t.box[c, 3:], st.pos[s, :3].max(0))
        mm, xx = m[s], x[s]
        cc = (mm[:, None] * xx).sum(0) / mm.sum()
        rr = xx - cc
        qq = np.einsum("i,ij,ik->jk", mm, rr, rr)
        assert np.allclose(t.mom64[c, 0], mm.sum(), rtol=1e-13)
        assert np.allclose(t.mom64[c, 1:4], cc, atol=1e-12)
        assert np.allclose(t.mom64[c, 4:], [qq[0, 0], qq[1, 1], qq[2, 2], qq[0, 1], qq[0, 2], qq[1, 2]],
                           rtol=1e-9, atol=1e-16)


def test_parallel_axis_identity_at_every_node():
    st, _ = _state("c3", 20000)
    t = st.tree
    idx = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    for c in np.nonzero(t.nchild > 0)[0]:
        ch = np.arange(t.child_begin[c], t.child_begin[c] + t.nchild[c])
        Mc, cc, Qc = t.mom64[ch, 0], t.mom64[ch, 1:4], t.mom64[ch, 4:]
        M = Mc.sum()
        com = (Mc[:, None] * cc).sum(0) / M
        d = cc - com
        Q = np.array([Qc[:, k].sum() + (Mc * d[:, a] * d[:, b]).sum() for k, (a, b) in enumerate(idx)])
        assert abs(t.mom64[c, 0] - M) <= 1e-14 * M
        assert np.allclose(t.mom64[c, 1:4], com, atol=1e-13)
        assert np.allclose(t.mom64[c, 4:], Q, rtol=1e-10, atol=1e-18)


# ---------------------------------------------------------------- P7: the p-c formula on a hand-made tree
def _hand_tree(src, tgt):
    """Root node with two leaf children: A = the source particles, B = the single target.

    Bypasses keys/sort/tree so that the moments (O8), the MAC (O9) and the p-c formula (O10) are
    exercised on a topology fixed by hand.
    """
    na = src.shape[0]
    pos = np.concatenate([src, tgt]).astype(np.float32)
    n = pos.shape[0]
    lo = np.zeros(22, np.int64); lo[1] = 1; lo[2:] = 3
    t = oracle.Tree(n, lo, np.array([0, 1, 1], np.int32), np.array([0, 0, 7], np.uint64),
                    np.array([0, 0, na], np.int64), np.array([n, na, n - na], np.int64),
                    np.array([1, -1, -1], np.int64), np.array([2, 0, 0], np.int32), np.array([-1, 0, 0], np.int64))
    t.gcell = np.array([2], np.int64); t.gbegin = np.array([na], np.int64); t.gcount = np.array([n - na], np.int64)
    oracle.moments(t, pos)
    return t, pos


def test_pc_closed_form_two_masses_on_axis():
    # two equal masses m at (+-s, 0, 0), target on the axis at R: a_x = -(m/(R-s)^2 + m/(R+s)^2)
    # = -(2m/R^2)(1 + 3 s^2/R^2 + 5 s^4/R^4 + ...); monopole + quadrupole keeps the first two terms.
    m, s, R = 0.5, 0.125, 8.0
    src = np.array([[-s, 0, 0, m], [s, 0, 0, m]])
    t, pos = _hand_tree(src, np.array([[R, 0, 0, 1.0]]))
    assert np.allclose(t.mom64[1], [2 * m, 0, 0, 0, 2 * m * s * s, 0, 0, 0, 0, 0], atol=1e-15)
    r = oracle.walk_forces(t, pos, theta=0.5, eps=0.0)
    assert r["npc"][0] == 1 and r["npp"][0] == 1          # cell A accepted, own leaf opened
    ax, ay, az, phi = r["accpot"][2]
    quad = -(2 * m / R ** 2) * (1 + 3 * s ** 2 / R ** 2)
    exact = -(m / (R - s) ** 2 + m / (R + s) ** 2)
    assert abs(ax - quad) < 1e-15 and ay == 0 and az == 0
    assert abs(ax - exact) / abs(exact) < 6 * (s / R) ** 4   # next term is 5 s^4 / R^4
    phi_quad = -(2 * m / R) * (1 + s ** 2 / R ** 2)
    assert abs(phi - phi_quad) < 1e-15
    # off axis (target on y): a_y = -2 m R / (R^2+s^2)^(3/2) = -(2m/R^2)(1 - 3 s^2 / (2 R^2) + ...)
    t, pos = _hand_tree(src, np.array([[0, R, 0, 1.0]]))
    r = oracle.walk_forces(t, pos, theta=0.5, eps=0.0)
    ax, ay, az, phi = r["accpot"][2]
    assert abs(ay + (2 * m / R ** 2) * (1 - 1.5 * s ** 2 / R ** 2)) < 1e-15 and ax == 0 and az == 0
    assert abs(phi + (2 * m / R) * (1 - 0.5 * s ** 2 / R ** 2)) < 1e-15


@pytest.mark.parametrize("eps", [0.0, 0.05, 0.2])
def test_pc_error_falls_as_cube_of_size_over_distance(eps):
    rng = np.random.default_rng(5)
    s = 0.1
    src = np.concatenate([rng.uniform(-s, s, (16, 3)), rng.uniform(0.5, 1.5, (16, 1))], axis=1).astype(np.float32)
    dirn = np.array([0.3, -0.5, 0.81]); dirn /= np.linalg.norm(dirn)
    errs, Rs = [], [1.0, 2.0, 4.0, 8.0]
    for R in Rs:
        t, pos = _hand_tree(src, np.array([np.append(R * dirn, 1.0)]))
        r = oracle.walk_forces(t, pos, theta=0.9, eps=eps)
        assert r["npc"][0] == 1
        d = oracle.direct(pos, eps)[16]
        got = r["accpot"][16]
        errs.append((np.linalg.norm(got[:3] - d[:3]) / np.linalg.norm(d[:3]), abs(got[3] - d[3]) / abs(d[3])))
    errs = np.array(errs)
    for k in range(len(Rs) - 1):   # doubling R must cut the relative error by ~8 (octupole term); demand > 5
        assert errs[k, 0] / errs[k + 1, 0] > 5.0, errs
        assert errs[k, 1] / errs[k + 1, 1] > 5.0, errs
    assert errs[-1, 0] < 5e-6


def test_single_particle_cell_is_particle_particle():
    src = np.array([[0.25, -0.5, 0.125, 0.75]])
    t, pos = _hand_tree(src, np.array([[3.0, 1.0, -2.0, 1.0]]))
    for eps in (0.0, 0.3):
        r = oracle.walk_forces(t, pos, theta=0.5, eps=eps)
        assert r["npc"][0] == 1
        d = oracle.direct(pos, eps)[1]
        assert np.allclose(r["accpot"][1], d, rtol=1e-15, atol=0)


# ---------------------------------------------------------------- P8: walk + forces vs brute force
def test_theta_to_zero_reproduces_direct_sum():
    st, _ = _state("c1", 2048)
    d = oracle.direct(st.pos, 0.01)
    oracle.compute_forces(st, theta=1e-6, eps=0.01)
    assert np.allclose(st.accpot, d, rtol=1e-12, atol=1e-13)
    # every particle appears either as a particle or as a single-particle cell
    assert np.all(st.npc + st.npp == st.tree.n)


def test_tree_error_small_and_monotone_in_theta():
    st, _ = _state("c1", 4096)
    d = oracle.direct(st.pos, 0.0)
    med = []
    for th in (0.8, 0.6, 0.4, 0.2):
        oracle.compute_forces(st, theta=th, eps=0.0)
        med.append(np.median(_relerr(st.accpot, d)))
    assert all(med[i] > med[i + 1] for i in range(3)), med
    assert med[0] < 3e-3 and med[-1] < 3e-5, med


def test_uniform_cube_vs_direct():
    st, prm = _state("c3", 3000)
    d = oracle.direct(st.pos, prm["eps"])
    oracle.compute_forces(st, theta=prm["theta"], eps=prm["eps"])
    e = _relerr(st.accpot, d)
    assert np.median(e) < 2e-3 and e.max() < 0.2
    assert np.max(np.abs(st.accpot[:, 3] - d[:, 3]) / np.abs(d[:, 3])) < 1e-3


# ---------------------------------------------------------------- P9: MAC geometry
def test_no_accepted_cell_contains_a_group_particle():
    st, _ = _state("c1", 8192)
    t = st.tree
    for g in range(0, t.ngroups, 23):
        r = oracle.walk_forces(t, st.pos, theta=1.0, eps=0.01, sel=[g], forces=False, want_lists=True)
        b, e = t.gbegin[g], t.gbegin[g] + t.gcount[g]
        cb, ce = t.pbegin[r["cells"]], t.pbegin[r["cells"]] + t.pcount[r["cells"]]
        assert not np.any((cb < e) & (ce > b))
        # lists cover every particle exactly once
        assert t.pcount[r["cells"]].sum() + t.pcount[r["leaves"]].sum() == t.n
        assert r["npp"][g] == t.pcount[r["leaves"]].sum() and r["npc"][g] == r["cells"].size


# ---------------------------------------------------------------- P10 / P11: potential, momentum
def test_plummer_potential_and_energies():
    st, _ = _state("c1", 16384)
    oracle.compute_forces(st, theta=0.5, eps=0.01)
    a = bh_inputs.PLUMMER_A
    p = st.pos.astype(np.float64)
    r = np.linalg.norm(p[:, :3], axis=1)
    phi_an = -1.0 / np.sqrt(r * r + a * a)
    rel = np.abs(st.accpot[:, 3] - phi_an) / np.abs(phi_an)
    assert np.median(rel) < 0.02 and np.percentile(rel, 99) < 0.12
    W = 0.5 * np.sum(p[:, 3] * st.accpot[:, 3])
    K = 0.5 * np.sum(p[:, 3] * np.sum(st.vel[:, :3].astype(np.float64) ** 2, axis=1))
    assert abs(W + 0.5) < 0.02 and abs(K - 0.25) < 0.01      # -3 pi M^2 / (32 a) = -1/2; virial K = 1/4
    # acceleration magnitude against the analytic field M r / (r^2 + a^2)^(3/2), outside the noisy core
    sel = r > 0.5
    ar = -np.sum(st.accpot[:, :3] * p[:, :3], axis=1) / r
    an = r / np.power(r * r + a * a, 1.5)
    assert np.median(np.abs(ar[sel] - an[sel]) / an[sel]) < 0.03


def test_momentum_conservation():
    st, _ = _state("c1", 4096)
    m = st.pos[:, 3].astype(np.float64)
    d = oracle.direct(st.pos, 0.01)
    scale = np.sum(m * np.linalg.norm(d[:, :3], axis=1))
    assert np.linalg.norm((m[:, None] * d[:, :3]).sum(0)) / scale < 1e-14
    oracle.compute_forces(st, theta=0.75, eps=0.01)
    assert np.linalg.norm((m[:, None] * st.accpot[:, :3]).sum(0)) / scale < 2e-4


# ---------------------------------------------------------------- P12 / P13: leapfrog
def _energy(st):
    m = st.pos[:, 3].astype(np.float64)
    K = 0.5 * np.sum(m * np.sum(st.vel[:, :3].astype(np.float64) ** 2, axis=1))
    W = 0.5 * np.sum(m * st.accpot[:, 3])
    return K + W


def test_two_body_circular_orbit():
    # two unit masses, separation 2 -> each at radius 1 feels a = 1/4: v = 1/2, period 4 pi
    pm = np.array([[1, 0, 0, 1], [-1, 0, 0, 1]], np.float32)
    v = np.array([[0, 0.5, 0, 0], [0, -0.5, 0, 0]], np.float32)
    steps = 256
    dt = 4 * math.pi / steps
    st = oracle.compute_forces(oracle.tree_build(pm, v), 0.5, 0.0)
    assert np.allclose(st.accpot[np.argsort(st.ids)], [[-0.25, 0, 0, -0.5], [0.25, 0, 0, -0.5]], atol=1e-15)
    e0 = _energy(st)
    rmin, rmax = 1.0, 1.0
    for _ in range(steps):
        st = oracle.leapfrog_step(st, 0.5, 0.0, dt)
        rr = np.linalg.norm(st.pos[:, :3], axis=1)
        rmin, rmax = min(rmin, rr.min()), max(rmax, rr.max())
    o = np.argsort(st.ids)
    assert np.allclose(st.pos[o, :3], pm[:, :3], atol=3e-3)        # back at the start after one period
    assert rmax - rmin < 2e-3 and abs(_energy(st) - e0) < 1e-5


def test_leapfrog_reversible_and_second_order():
    pm, v, _ = bh_inputs.make("c1", n=512)
    st0 = oracle.compute_forces(oracle.tree_build(pm, v), 1e-6, 0.05)     # direct-sum forces
    # reversibility: n steps, flip v, n steps -> start (up to float32 rounding of x, v)
    st = st0
    for _ in range(4):
        st = oracle.leapfrog_step(st, 1e-6, 0.05, 1 / 64)
    st.vel = -st.vel
    for _ in range(4):
        st = oracle.leapfrog_step(st, 1e-6, 0.05, 1 / 64)
    o, o0 = np.argsort(st.ids), np.argsort(st0.ids)
    assert np.max(np.abs(st.pos[o, :3] - st0.pos[o0, :3])) < 2e-5
    assert np.max(np.abs(-st.vel[o, :3] - st0.vel[o0, :3])) < 2e-5
    # energy error over a fixed time span scales as dt^2 (softening 0.2 so that dt resolves every encounter)
    sa = oracle.compute_forces(oracle.tree_build(pm, v), 1e-6, 0.2)
    errs = []
    for nst in (4, 8, 16):
        st = sa
        for _ in range(nst):
            st = oracle.leapfrog_step(st, 1e-6, 0.2, 0.25 / nst)
        errs.append(abs(_energy(st) - _energy(sa)))
    assert 3.0 < errs[0] / errs[1] < 5.5 and 3.0 < errs[1] / errs[2] < 5.5, errs


def test_energy_drift_c1_is_small():
    pm, v, prm = bh_inputs.make("c1", n=4096)
    st = oracle.compute_forces(oracle.tree_build(pm, v), prm["theta"], prm["eps"])
    e0 = _energy(st)
    for _ in range(4):
        st = oracle.leapfrog_step(st, prm["theta"], prm["eps"], prm["dt"])
    assert abs((_energy(st) - e0) / e0) < 2e-4      # context: the paper's merger, ~1e-4 (Table 2)


# ---------------------------------------------------------------- P14: determinism
def test_deterministic_across_runs():
    st, prm = _state("c1", 8192)
    a = oracle.walk_forces(st.tree, st.pos, 0.75, 0.01)
    b = oracle.walk_forces(st.tree, st.pos, 0.75, 0.01)
    assert np.array_equal(a["accpot"], b["accpot"]) and np.array_equal(a["npc"], b["npc"])


# ---------------------------------------------------------------- minimum-distance MAC (reading A28)
def _mindist_accept_np(gbox, cbox, theta):
    """A28 restated in numpy float32: per-axis gap between two boxes, d2 by fused multiply-adds, accept iff d2 > (l / theta)^2."""
    f = np.float32
    d = np.maximum(np.maximum(gbox[:3] - cbox[3:], cbox[:3] - gbox[3:]), f(0)).astype(np.float32)
    d2 = f(np.float64(d[0]) * np.float64(d[0]))                      # one rounding: the product of two floats is exact in double
    d2 = f(np.float64(d[1]) * np.float64(d[1]) + np.float64(d2))     # fmaf: exact product + addend, one rounding
    d2 = f(np.float64(d[2]) * np.float64(d[2]) + np.float64(d2))
    l = np.max((cbox[3:] - cbox[:3]).astype(np.float32))
    r = f(l / f(theta))
    return d2 > f(r * r)


def test_mindist_mac_lists_equal_a_walk_written_from_the_definition():
    st, _ = _state("c1", 3000)
    t = st.tree
    theta = 0.6
    for g in range(0, t.ngroups, 7):
        r = oracle.walk_forces(t, st.pos, theta=theta, eps=0.01, sel=[g], forces=False, want_lists=True, mac_kind=oracle.MAC_MINDIST)
        cells, leaves, todo = [], [], [0]
        while todo:
            c = todo.pop()
            if _mindist_accept_np(t.gbox[g], t.box[c], theta):
                cells.append(c)
            elif t.nchild[c] == 0:
                leaves.append(c)
            else:
                todo.extend(range(t.child_begin[c], t.child_begin[c] + t.nchild[c]))
        assert sorted(cells) == sorted(r["cells"].tolist()) and sorted(leaves) == sorted(r["leaves"].tolist())
        # an accepted cell's box is strictly separated from the group's box, and the lists cover every particle once
        for c in cells:
            gap = np.maximum(np.maximum(t.gbox[g][:3] - t.box[c][3:], t.box[c][:3] - t.gbox[g][3:]), 0)
            assert np.any(gap > 0)
        assert t.pcount[cells].sum() + t.pcount[leaves].sum() == t.n


def test_mindist_mac_limits_and_accuracy():
    st, _ = _state("c1", 4096)
    d = oracle.direct(st.pos, 0.01)
    # theta -> 0: the direct sum
    oracle.compute_forces(st, theta=1e-6, eps=0.01, mac_kind=oracle.MAC_MINDIST)
    assert _relerr(st.accpot, d).max() < 1e-12          # (accepted cells are single particles: l = 0, exact)
    # same theta: opens more than Eq.1 and is more accurate (the paper: smaller error, more interactions, L129)
    oracle.compute_forces(st, theta=0.75, eps=0.01)
    n0, e0 = st.npc.sum() + st.npp.sum(), _relerr(st.accpot, d)
    oracle.compute_forces(st, theta=0.75, eps=0.01, mac_kind=oracle.MAC_MINDIST)
    n1, e1 = st.npc.sum() + st.npp.sum(), _relerr(st.accpot, d)
    assert n1 > n0 and np.median(e1) < np.median(e0) and np.quantile(e1, 0.99) < np.quantile(e0, 0.99)
    # r2_open is (l / theta)^2 with l the longest side of the tight box
    l = (st.tree.box[:, 3:] - st.tree.box[:, :3]).max(axis=1).astype(np.float32)
    r = (l / np.float32(0.75)).astype(np.float32)
    assert np.array_equal(st.mac[:, 2], (r * r).astype(np.float32))


# ---------------------------------------------------------------- Eq.1 (Fig.5): the VALUE of l, delta, r_open
def _two_particle_cell_case(B, mB, xt_x, theta=0.5):
    """A = (0,0,0) with mass 1 and B with mass mB form one leaf (nleaf = ncrit = 2); the target T sits alone in another
    cell, level with the leaf's centre of mass in y and z, so that d(group box, com) = T.x - com.x.  Returns
    (mac row of the leaf {A, B}, n_pc of T's group, n_pp of T's group)."""
    com = np.array(B[:3]) * mB / (1.0 + mB)
    pm = np.array([[0, 0, 0, 1.0], [B[0], B[1], B[2], mB], [xt_x, com[1], com[2], 1.0]], np.float32)
    st = oracle.tree_build(pm, nleaf=2, ncrit=2)
    t = st.tree
    assert t.ncells == 3 and t.ngroups == 2 and list(t.pcount) == [3, 2, 1] and list(t.gcount) == [2, 1]
    oracle.compute_forces(st, theta=theta, eps=0.0)
    return st.mac[1], int(st.npc[1]), int(st.npp[1])


def test_eq1_opening_radius_closed_form_and_flip_at_the_threshold():
    """Hand-built cells whose l, delta and r_open are exact binary fractions known in closed form (Eq.1: d > l/theta + delta,
    l = cell size, delta = |geometric centre - centre of mass|), and a target one ulp on either side of
    the threshold.  A wrong delta (halved, dropped, measured from a box corner), a wrong sign or a wrong l fails here."""
    f = np.float32
    # (1) on an axis: box [0,1], l = 1, centre 0.5, com = 0.75, delta = 0.25; theta = 0.5: r_open = 2.25, r2_open = 5.0625
    mac, npc, npp = _two_particle_cell_case((1, 0, 0), 3.0, 3.0)           # d = 3 - 0.75 = 2.25 exactly: NOT accepted (strict, A16)
    assert tuple(mac) == (f(1.0), f(0.25), f(5.0625))
    assert (npc, npp) == (0, 3)                                             # leaf {A,B} opened (2) + own leaf (1)
    mac, npc, npp = _two_particle_cell_case((1, 0, 0), 3.0, np.nextafter(f(3.0), f(4.0)))
    assert tuple(mac) == (f(1.0), f(0.25), f(5.0625)) and (npc, npp) == (1, 1)    # one ulp further: accepted
    # (2) off-axis offset: B = (2,2,1), masses 1:3 -> box [0,2]x[0,2]x[0,1], l = 2, centre (1,1,.5), com = (1.5,1.5,.75),
    #     u = (.5,.5,.25), delta = sqrt(.5625) = .75; theta = 0.5: r_open = 4.75, r2_open = 22.5625; threshold T.x = 6.25
    mac, npc, npp = _two_particle_cell_case((2, 2, 1), 3.0, 6.25)
    assert tuple(mac) == (f(2.0), f(0.75), f(22.5625)) and (npc, npp) == (0, 3)
    mac, npc, npp = _two_particle_cell_case((2, 2, 1), 3.0, np.nextafter(f(6.25), f(7.0)))
    assert (npc, npp) == (1, 1)
    # (3) equal masses: com = centre, delta = 0 exactly: r_open = l / theta alone (theta = 0.25: 4, r2 = 16; threshold 4.5)
    mac, npc, npp = _two_particle_cell_case((1, 0, 0), 1.0, 4.5, theta=0.25)
    assert tuple(mac) == (f(1.0), f(0.0), f(16.0)) and (npc, npp) == (0, 3)
    mac, npc, npp = _two_particle_cell_case((1, 0, 0), 1.0, np.nextafter(f(4.5), f(5.0)), theta=0.25)
    assert (npc, npp) == (1, 1)


def _eq1_accept_np(gbox, com, r2open):
    """O9 restated in numpy float32: per-axis distance from the group's box to the centre of mass, d2 by fused multiply-adds."""
    f = np.float32
    d = np.maximum(np.maximum(gbox[:3] - com, com - gbox[3:]), f(0)).astype(np.float32)
    d2 = f(np.float64(d[0]) * np.float64(d[0]))                      # one rounding: the product of two floats is exact in double
    d2 = f(np.float64(d[1]) * np.float64(d[1]) + np.float64(d2))     # fmaf: exact product + addend, one rounding
    d2 = f(np.float64(d[2]) * np.float64(d[2]) + np.float64(d2))
    return d2 > r2open


def test_eq1_mac_columns_and_lists_equal_a_walk_written_from_the_definition():
    """The Eq.1 twin of the minimum-distance pin: l, delta, r2_open of EVERY cell from the tight box and the fp32 centre of
    mass in numpy float32 (array_equal on all three columns), and the lists of a root-to-leaf walk with that test."""
    st, _ = _state("c1", 3000)
    t = st.tree
    theta = np.float32(0.6)
    r = oracle.walk_forces(t, st.pos, theta=float(theta), eps=0.01, sel=[0], forces=False)
    mac = r["mac"]
    com = t.mom64[:, 1:4].astype(np.float32)
    bmin, bmax = t.box[:, :3], t.box[:, 3:]
    l = (bmax - bmin).astype(np.float32).max(axis=1)
    gc = (np.float32(0.5) * (bmin + bmax).astype(np.float32)).astype(np.float32)
    u = (com - gc).astype(np.float32)
    uu = (u * u).astype(np.float32)
    s2 = ((uu[:, 0] + uu[:, 1]).astype(np.float32) + uu[:, 2]).astype(np.float32)
    delta = np.sqrt(s2).astype(np.float32)
    ropen = ((l / theta).astype(np.float32) + delta).astype(np.float32)
    assert np.array_equal(mac[:, 0], l) and np.array_equal(mac[:, 1], delta)
    assert np.array_equal(mac[:, 2], (ropen * ropen).astype(np.float32))
    assert np.count_nonzero(delta) > 0.5 * t.ncells                 # the offset term is exercised by every cell with more than one particle
    for g in range(0, t.ngroups, 7):
        r = oracle.walk_forces(t, st.pos, theta=float(theta), eps=0.01, sel=[g], forces=False, want_lists=True)
        cells, leaves, todo = [], [], [0]
        while todo:
            c = todo.pop()
            if _eq1_accept_np(t.gbox[g], com[c], mac[c, 2]):
                cells.append(c)
            elif t.nchild[c] == 0:
                leaves.append(c)
            else:
                todo.extend(range(t.child_begin[c], t.child_begin[c] + t.nchild[c]))
        assert sorted(cells) == sorted(r["cells"].tolist()) and sorted(leaves) == sorted(r["leaves"].tolist())
