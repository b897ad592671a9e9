"""Pins for the oracle's block time-step scheme (reading A29), no GPU.

Closed forms for the time-step criterion, the invariants of commensurate power-of-two steps, the one-rung case against
the shared-step leapfrog, second-order convergence on a two-body orbit whose bodies take unequal steps, and the energy
of a Plummer sphere over a macro-step."""
import numpy as np

import bh_inputs
import oracle


def test_rung_criterion_closed_forms_and_thresholds():
    f = np.float32
    acc = np.zeros((6, 4), np.float32)
    acc[0, 0] = 4.0                      # tau = 0.5 sqrt(0.01 / 4) = 0.025: 1/16, 1/32 are too long, 1/64 fits -> rung 2
    acc[1, :3] = (0.0, 3.0, 4.0)          # |a| = 5: tau = 0.5 sqrt(0.002) = 0.02236: 1/64 = 0.0156 fits -> rung 2
    acc[2, 2] = 0.25                      # tau = 0.5 sqrt(0.04) = 0.1 >= 1/16 -> rung 0
    acc[3, 1] = 1e6                       # tau = 5e-5: not even dt_max / 2^5 fits -> the deepest rung
    acc[4] = 0.0                          # |a| = 0: tau = inf -> rung 0
    acc[5, 0] = 0.64                      # tau = 0.5 sqrt(0.015625) = 0.0625 = dt_max exactly: "<=" -> rung 0
    r = oracle.rungs(acc, None, 0.01, 0.5, 1.0 / 16, 5, 0)
    assert list(r) == [2, 2, 0, 5, 0, 0]
    # one ulp above the threshold acceleration: the step no longer fits
    acc[5, 0] = np.nextafter(f(0.64), f(1.0))
    assert oracle.rungs(acc, None, 0.01, 0.5, 1.0 / 16, 5, 0)[5] == 1
    # a longer step may only start at a time that is a multiple of it: at tick 4 of R = 5 (step(r) = 2^(5-r) ticks), rung >= 3
    r = oracle.rungs(acc, None, 0.01, 0.5, 1.0 / 16, 5, 4)
    assert list(r) == [3, 3, 3, 5, 3, 3]
    assert list(oracle.rungs(acc, None, 0.01, 0.5, 1.0 / 16, 5, 32)) == [2, 2, 0, 5, 0, 1]      # a multiple of every step
    # only the active particles get a new rung
    out = np.full(6, 9, np.uint8)
    oracle.rungs(acc, np.array([1, 0, 0, 0, 0, 1], np.uint8), 0.01, 0.5, 1.0 / 16, 5, 0, out=out)
    assert list(out) == [2, 9, 9, 9, 9, 1]


def _block_state(n=2048, R=3, eta=0.2, seed=None, theta=0.5, eps=0.02, dt_max=1.0 / 16):
    pm, v, _ = bh_inputs.make("c1", n=n, seed=seed)
    st = oracle.compute_forces(oracle.tree_build(pm, v), theta, eps)
    return oracle.block_init(st, eps, eta, dt_max, R), theta, eps


def test_times_stay_commensurate_and_everybody_is_updated():
    bs, theta, eps = _block_state(R=4)
    assert len(set(bs.rung)) >= 3                       # the criterion spreads a Plummer sphere over several rungs
    seen = np.zeros(bs.tree.n, bool)
    last = 0
    while bs.now < 16:                                   # one macro-step = 2^R ticks
        bs = oracle.block_step(bs, theta, eps)
        step = (1 << (bs.R - bs.rung.astype(np.int64)))
        assert bs.now > last and np.all(bs.tick % step == 0) and np.all(bs.tick <= bs.now)
        assert np.array_equal(bs.active != 0, bs.tick == bs.now)          # exactly the due particles were moved to `now`
        seen |= bs.active != 0
        last = bs.now
    assert bs.now == 16 and seen.all() and np.all(bs.tick == 16)          # the longest step ends at the macro-step: all synchronised


def test_one_rung_is_the_shared_step_leapfrog():
    """R = 0: every particle is active in every step; the predictor-corrector is algebraically kick-drift-kick (A21)."""
    pm, v, _ = bh_inputs.make("c1", n=1024, seed=3)
    theta, eps, dt = 0.4, 0.05, 1.0 / 64
    st = oracle.compute_forces(oracle.tree_build(pm, v), theta, eps)
    bs = oracle.block_init(st, eps, 1e9, dt, 0)
    assert np.all(bs.rung == 0)
    ref = st
    for _ in range(4):
        bs = oracle.block_step(bs, theta, eps)
        ref = oracle.leapfrog_step(ref, theta, eps, dt)
    o, o2 = np.argsort(bs.ids), np.argsort(ref.ids)
    assert np.max(np.abs(bs.pos[o, :3] - ref.pos[o2, :3])) < 2e-5       # (the cells of bs are not rebuilt: lists differ slightly)
    assert np.max(np.abs(bs.vel[o, :3] - ref.vel[o2, :3])) < 2e-4


def _two_body(eta, R=6, T=4.0, dt_max=1.0 / 8):
    """Masses 1 and 0.1 on a bound eccentric orbit: the light body sees ten times the acceleration and takes shorter steps.
    Returns the largest relative energy error at the synchronised times, and the rungs that occurred."""
    pm = np.array([[0, 0, 0, 1.0], [1.0, 0, 0, 0.1]], np.float32)
    vel = np.array([[0, -0.09, 0, 0], [0, 0.9, 0, 0]], np.float32)
    st = oracle.compute_forces(oracle.tree_build(pm, vel, nleaf=1, ncrit=1), 1e-6, 0.0)

    def energy(pos, vel_):
        p, w = pos.astype(np.float64), vel_.astype(np.float64)
        d = np.linalg.norm(p[0, :3] - p[1, :3])
        return 0.5 * (p[0, 3] * (w[0, :3] ** 2).sum() + p[1, 3] * (w[1, :3] ** 2).sum()) - p[0, 3] * p[1, 3] / d

    bs = oracle.block_init(st, 0.05, eta, dt_max, R)
    e0 = energy(bs.pos, bs.vel)
    worst, rungs_seen, mixed = 0.0, set(), False
    while bs.now < int(T / dt_max) << R:
        bs = oracle.block_step(bs, 1e-6, 0.0)
        rungs_seen |= set(int(x) for x in bs.rung)
        mixed |= bs.rung[0] != bs.rung[1]
        if np.all(bs.tick == bs.now):
            worst = max(worst, abs(energy(bs.pos, bs.vel) - e0) / abs(e0))
    assert np.all(bs.tick == bs.now)
    return worst, rungs_seen, mixed


def test_two_body_orbit_with_unequal_steps_converges():
    """The predictor-corrector with individually chosen, changing steps is not time-symmetric: the energy error falls at
    least linearly with eta (second order needs fixed steps: the one-rung case above)."""
    e = {eta: _two_body(eta) for eta in (0.2, 0.1, 0.05)}
    assert all(v[2] for v in e.values())                     # the bodies really were on different rungs
    assert e[0.2][0] < 0.05 and e[0.05][0] < 0.01
    assert e[0.2][0] / e[0.1][0] > 1.7 and e[0.1][0] / e[0.05][0] > 1.7, e


def test_energy_over_a_macro_step_of_a_plummer_sphere():
    bs, theta, eps = _block_state(n=4096, R=3, eta=0.1, seed=11, theta=0.4, eps=0.05)

    def energy(b):
        # synchronised state: potential from a fresh direct sum
        d = oracle.direct(b.pos, eps)
        m = b.pos[:, 3].astype(np.float64)
        return 0.5 * np.sum(m * np.sum(b.vel[:, :3].astype(np.float64) ** 2, axis=1)) + 0.5 * np.sum(m * d[:, 3])

    e0 = energy(bs)
    nsteps = 0
    while bs.now < 8:
        bs = oracle.block_step(bs, theta, eps)
        nsteps += 1
    assert np.all(bs.tick == 8) and nsteps >= 4
    assert abs((energy(bs) - e0) / e0) < 2e-4
