"""Seeded synthetic initial conditions for the Barnes-Hut pipeline.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_1106_1900_b200/``).  It holds none of the method's arithmetic: it
only draws particles.  The paper's performance workload is Plummer spheres
(section 4.1); the remaining shapes are BASELINE.json configs 3-5.
The galaxy-merger initial conditions of PAPER.md:208-214 are not available and
are not reproduced.

Every generator draws in float64 from ``numpy.random.Generator(Philox(seed))``
and casts to float32 exactly once.  Layout: ``pos_mass`` is ``float32[N,4]``
(x, y, z, m) and ``vel`` is ``float32[N,4]`` (vx, vy, vz, 0), the same layout
both the oracle and the CUDA library take.
"""
from __future__ import annotations

import math

import numpy as np

SEEDS = {"c1": 11061901, "c2": 11061902, "c3": 11061903, "c4": 11061904, "c5": 11061905}
PLUMMER_A = 3.0 * math.pi / 16.0  # N-body units: M = 1, E = -1/4  (BASELINE.json configs 1-2)


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(int(seed)))


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    """n unit vectors, uniform on the sphere (float64[n,3])."""
    cz = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * math.pi, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return np.stack([s * np.cos(ph), s * np.sin(ph), cz], axis=1)


def _plummer_q_table(npts: int = 4096):
    """Cumulative table of g(q) ~ q^2 (1-q^2)^(7/2) on [0,1] (speed / escape speed)."""
    q = np.linspace(0.0, 1.0, npts)
    g = q * q * np.power(np.maximum(0.0, 1.0 - q * q), 3.5)
    c = np.concatenate([[0.0], np.cumsum(0.5 * (g[1:] + g[:-1]) * np.diff(q))])
    return q, c / c[-1]


def _plummer64(rng, n, mass, a, umax=0.999):
    """Plummer sphere in float64: (pos[n,3], vel[n,3], m[n])."""
    u = rng.uniform(0.0, umax, n)
    u = np.maximum(u, 1e-300)
    r = a / np.sqrt(np.power(u, -2.0 / 3.0) - 1.0)
    pos = r[:, None] * _isotropic(rng, n)
    qt, ct = _plummer_q_table()
    q = np.interp(rng.uniform(0.0, 1.0, n), ct, qt)
    vesc = math.sqrt(2.0 * mass) * np.power(r * r + a * a, -0.25)
    vel = (q * vesc)[:, None] * _isotropic(rng, n)
    m = np.full(n, mass / n)
    return pos, vel, m


def _pack(pos, vel, m):
    n = pos.shape[0]
    pm = np.empty((n, 4), dtype=np.float32)
    pm[:, :3] = pos
    pm[:, 3] = m
    v = np.zeros((n, 4), dtype=np.float32)
    v[:, :3] = vel
    return pm, v


def plummer(n: int, seed: int = SEEDS["c2"], mass: float = 1.0, a: float = PLUMMER_A,
            umax: float = 0.999):
    """Plummer sphere, truncated at the radius holding ``umax`` of the mass.

    Radius by inverse CDF r = a (u^(-2/3) - 1)^(-1/2), u ~ U(0, umax); isotropic direction;
    speed q * v_esc(r) with q from the tabulated CDF of q^2 (1-q^2)^(7/2); m = mass / n.
    """
    rng = _rng(seed)
    return _pack(*_plummer64(rng, n, mass, a, umax))


def uniform_cube(n: int, seed: int = SEEDS["c3"], half: float = 1.0):
    """Uniform in [-half, half]^3, equal masses summing to 1, zero velocities (config 3)."""
    rng = _rng(seed)
    pos = rng.uniform(-half, half, (n, 3))
    return _pack(pos, np.zeros((n, 3)), np.full(n, 1.0 / n))


def _invert_monotone(f, lo, hi, y, npts=65536):
    x = np.linspace(lo, hi, npts)
    return np.interp(y, f(x), x)


def galaxy3(n: int = 16_777_216, seed: int = SEEDS["c4"]):
    """Three-component galaxy (config 4): NFW halo, Hernquist bulge, exponential disk.

    Particle split 10 000 000 : 2 000 000 : remainder (4 777 216 at the configured n),
    scaled proportionally for other n.  Velocities: disk tangential sqrt(M(<r)/r) in the
    spherically averaged total mass; halo and bulge isotropic Gaussian with the dispersion
    sqrt(M(<r)/(3 r)) (a plain stand-in for the Jeans solution: equilibrium quality does
    not matter for a 2-step throughput measurement, only determinism does).
    """
    rng = _rng(seed)
    nh = int(round(n * 10_000_000 / 16_777_216))
    nb = int(round(n * 2_000_000 / 16_777_216))
    nd = n - nh - nb
    rs, mh = 10.0, 10.0
    ab, mb = 0.3, 0.3
    rd, zd, md = 1.0, 0.1, 1.0
    # halo: cumulative mass ~ ln(1+x) - x/(1+x), x = r/rs <= 20
    fh = lambda x: np.log1p(x) - x / (1.0 + x)
    xh = _invert_monotone(fh, 0.0, 20.0, rng.uniform(0.0, 1.0, nh) * fh(np.array(20.0)))
    ph = (xh * rs)[:, None] * _isotropic(rng, nh)
    # bulge: r = a sqrt(u) / (1 - sqrt(u)), u < 0.999
    ub = np.sqrt(rng.uniform(0.0, 0.999, nb))
    pb = (ab * ub / (1.0 - ub))[:, None] * _isotropic(rng, nb)
    # disk: cumulative 1 - (1+R) exp(-R), R <= 12 rd; z = zd * atanh(2u-1)
    fd = lambda x: 1.0 - (1.0 + x) * np.exp(-x)
    R = rd * _invert_monotone(fd, 0.0, 12.0, rng.uniform(0.0, 1.0, nd) * fd(np.array(12.0)))
    phi = rng.uniform(0.0, 2.0 * math.pi, nd)
    z = zd * np.arctanh(np.clip(2.0 * rng.uniform(0.0, 1.0, nd) - 1.0, -0.999999, 0.999999))
    pd = np.stack([R * np.cos(phi), R * np.sin(phi), z], axis=1)

    def menc(r):
        x = r / rs
        m_h = mh * fh(x) / fh(np.array(20.0))
        m_b = mb * (r / (r + ab)) ** 2
        m_d = md * fd(r / rd)
        return m_h + m_b + m_d

    def sigma(p):
        r = np.maximum(np.linalg.norm(p, axis=1), 1e-6)
        return np.sqrt(menc(r) / (3.0 * r))

    vh = rng.standard_normal((nh, 3)) * sigma(ph)[:, None]
    vb = rng.standard_normal((nb, 3)) * sigma(pb)[:, None]
    rr = np.maximum(np.linalg.norm(pd, axis=1), 1e-6)
    vc = np.sqrt(menc(rr) / rr)
    vd = np.stack([-vc * np.sin(phi), vc * np.cos(phi), np.zeros(nd)], axis=1)
    pos = np.concatenate([ph, pb, pd])
    vel = np.concatenate([vh, vb, vd])
    m = np.concatenate([np.full(nh, mh / nh), np.full(nb, mb / max(nb, 1)), np.full(nd, md / max(nd, 1))])
    return _pack(pos, vel, m)


def colliding_plummers(n_each: int = 16_777_216, seed: int = SEEDS["c5"], a: float = PLUMMER_A):
    """Two Plummer spheres (each M = 1), centres at x = -/+ 10 a, bulk v_x = +/- 0.25 (config 5)."""
    rng = _rng(seed)
    p1, v1, m1 = _plummer64(rng, n_each, 1.0, a)
    p2, v2, m2 = _plummer64(rng, n_each, 1.0, a)
    p1[:, 0] -= 10.0 * a
    p2[:, 0] += 10.0 * a
    v1[:, 0] += 0.25
    v2[:, 0] -= 0.25
    return _pack(np.concatenate([p1, p2]), np.concatenate([v1, v2]), np.concatenate([m1, m2]))


def make(config: str, n: int | None = None, seed: int | None = None):
    """Build the inputs of BASELINE.json config ``c1`` .. ``c5`` (optionally at another n / seed).

    Returns ``(pos_mass, vel, params)`` with params = dict(theta, eps, dt, steps).
    """
    if config == "c1":
        pm, v = plummer(n or 16_384, seed or SEEDS["c1"])
        return pm, v, dict(theta=0.75, eps=0.01, dt=1.0 / 64, steps=1)
    if config == "c2":
        pm, v = plummer(n or 1_048_576, seed or SEEDS["c2"])
        return pm, v, dict(theta=0.75, eps=0.01, dt=1.0 / 64, steps=4)
    if config == "c3":
        pm, v = uniform_cube(n or 4_194_304, seed or SEEDS["c3"])
        return pm, v, dict(theta=0.5, eps=0.005, dt=1.0 / 128, steps=2)
    if config == "c4":
        pm, v = galaxy3(n or 16_777_216, seed or SEEDS["c4"])
        return pm, v, dict(theta=0.4, eps=0.02, dt=1.0 / 256, steps=2)
    if config == "c5":
        pm, v = colliding_plummers((n or 33_554_432) // 2, seed or SEEDS["c5"])
        return pm, v, dict(theta=0.4, eps=0.01, dt=1.0 / 64, steps=10)
    raise ValueError(f"unknown config {config!r}")
