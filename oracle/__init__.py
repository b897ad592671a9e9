"""CPU oracle for the Barnes-Hut pipeline of arxiv/paper_1106_1900 -- TEST INFRASTRUCTURE.

Thin ctypes/numpy front end to ``bh_oracle.cpp`` (see that file's header for the citations and the
pins).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / --impl reference
legs may import this package; the product (``paper_1106_1900_b200``) never does, and this package
never imports the product.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field

import numpy as np

from .build import build as _build

NLEAF = 16
NCRIT = 64
MAXLEVEL = 20

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_build_tree.restype = C.c_int64
        _lib.orc_groups.restype = C.c_int64
        _lib.orc_dilate.restype = C.c_uint64
        _lib.orc_domain.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f32c(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == 4
    return a


def dilate(value: int, bits: int = 10) -> int:
    """PAPER.md:376 dilate: bit b of ``value`` moves to bit 3b."""
    return int(lib().orc_dilate(C.c_uint32(value), C.c_int32(bits)))


def domain(pos_mass):
    """O1.  Returns (lo float32[3], hi float32[3], e, ok)."""
    pm = _f32c(pos_mass)
    lo = np.zeros(3, np.float32)
    hi = np.zeros(3, np.float32)
    e = C.c_int32(0)
    rc = lib().orc_domain(C.c_int64(pm.shape[0]), _p(pm), _p(lo), _p(hi), C.byref(e))
    return lo, hi, int(e.value), rc == 0


def keys(pos_mass, lo, e):
    """O2 + O3: 60-bit Morton keys, uint64[N]."""
    pm = _f32c(pos_mass)
    lo = np.ascontiguousarray(lo, np.float32)
    out = np.empty(pm.shape[0], np.uint64)
    lib().orc_keys(C.c_int64(pm.shape[0]), _p(pm), _p(lo), C.c_int32(e), _p(out))
    return out


def sort_perm(k):
    """O4: stable ascending sort; perm[j] = input index of the j-th sorted key."""
    k = np.ascontiguousarray(k, np.uint64)
    perm = np.empty(k.shape[0], np.uint32)
    lib().orc_sort(C.c_int64(k.shape[0]), _p(k), _p(perm))
    return perm


@dataclass
class Tree:
    n: int
    level_offset: np.ndarray   # int64[22]
    level: np.ndarray          # int32[C]
    prefix: np.ndarray         # uint64[C]
    pbegin: np.ndarray         # int64[C]
    pcount: np.ndarray         # int64[C]
    child_begin: np.ndarray    # int64[C]  (-1 for leaves)
    nchild: np.ndarray         # int32[C]
    parent: np.ndarray         # int64[C]  (-1 for the root)
    gcell: np.ndarray = field(default=None)
    gbegin: np.ndarray = field(default=None)
    gcount: np.ndarray = field(default=None)
    mom64: np.ndarray = field(default=None)   # float64[C,10]
    box: np.ndarray = field(default=None)     # float32[C,6]
    gbox: np.ndarray = field(default=None)    # float32[G,6]

    @property
    def ncells(self):
        return int(self.level.shape[0])

    @property
    def ngroups(self):
        return int(self.gcell.shape[0])


def build_tree(sorted_keys, nleaf: int = NLEAF) -> Tree:
    """O6."""
    k = np.ascontiguousarray(sorted_keys, np.uint64)
    n = k.shape[0]
    L = lib()
    ncell = int(L.orc_build_tree(C.c_int64(n), _p(k), C.c_int32(nleaf), None, None, None, None, None,
                                 None, None, None))
    lo = np.zeros(MAXLEVEL + 2, np.int64)
    t = Tree(n, lo, np.empty(ncell, np.int32), np.empty(ncell, np.uint64), np.empty(ncell, np.int64),
             np.empty(ncell, np.int64), np.empty(ncell, np.int64), np.empty(ncell, np.int32),
             np.empty(ncell, np.int64))
    L.orc_build_tree(C.c_int64(n), _p(k), C.c_int32(nleaf), _p(t.level_offset), _p(t.level), _p(t.prefix),
                     _p(t.pbegin), _p(t.pcount), _p(t.child_begin), _p(t.nchild), _p(t.parent))
    return t


def make_groups(t: Tree, ncrit: int = NCRIT) -> Tree:
    """O7."""
    gc = np.empty(t.n, np.int64)
    gb = np.empty(t.n, np.int64)
    gn = np.empty(t.n, np.int64)
    g = int(lib().orc_groups(C.c_int64(t.ncells), _p(t.nchild), _p(t.pbegin), _p(t.pcount), _p(t.parent),
                             C.c_int32(ncrit), _p(gc), _p(gb), _p(gn)))
    t.gcell, t.gbegin, t.gcount = gc[:g].copy(), gb[:g].copy(), gn[:g].copy()
    return t


def moments(t: Tree, pos_sorted) -> Tree:
    """O8 (binary64 part) + group boxes."""
    pm = _f32c(pos_sorted)
    t.mom64 = np.zeros((t.ncells, 10), np.float64)
    t.box = np.zeros((t.ncells, 6), np.float32)
    lib().orc_moments(C.c_int64(t.ncells), _p(t.level_offset), _p(t.nchild), _p(t.child_begin),
                      _p(t.pbegin), _p(t.pcount), _p(pm), _p(t.mom64), _p(t.box))
    if t.gcell is not None:
        t.gbox = np.zeros((t.ngroups, 6), np.float32)
        lib().orc_group_boxes(C.c_int64(t.ngroups), _p(t.gbegin), _p(t.gcount), _p(pm), _p(t.gbox))
    return t


MAC_EQ1 = 0       # PAPER.md:125, Eq.1: d(group box, centre of mass) > l / theta + delta
MAC_MINDIST = 1   # PAPER.md:129 "minimal distance MAC [31]" (reading A28): d(group box, cell box) > l / theta


def cell_floats(t: Tree, theta: float, mac_kind: int = MAC_EQ1):
    """O8 float outputs: (mom32 float32[C,10], mac float32[C,3] = l, delta, r2_open)."""
    mom32 = np.empty((t.ncells, 10), np.float32)
    mac = np.empty((t.ncells, 3), np.float32)
    lib().orc_cell_floats(C.c_int64(t.ncells), _p(t.mom64), _p(t.box), C.c_float(theta), C.c_int32(mac_kind), _p(mom32), _p(mac))
    return mom32, mac


def walk_forces(t: Tree, pos_sorted, theta: float, eps: float, sel=None, forces: bool = True,
                want_lists: bool = False, mac_kind: int = MAC_EQ1):
    """O9 + O10 for the selected groups (default: all).

    Returns dict(npc int64[G], npp int64[G], accpot float64[N,4] or None, mom32, mac[, cells, leaves]).
    Entries of npc / npp / accpot outside the selection are -1 / NaN.
    """
    pm = _f32c(pos_sorted)
    mom32, mac = cell_floats(t, theta, mac_kind)
    G = t.ngroups
    sel = np.arange(G, dtype=np.int64) if sel is None else np.ascontiguousarray(sel, np.int64)
    npc = np.full(G, -1, np.int64)
    npp = np.full(G, -1, np.int64)
    acc = np.full((t.n, 4), np.nan, np.float64) if forces else None
    lc = ll = None
    if want_lists:
        assert sel.shape[0] == 1
        lc = np.full(t.ncells, -1, np.int64)
        ll = np.full(t.ncells, -1, np.int64)
    lib().orc_walk_forces(C.c_int64(t.n), _p(pm), _p(t.nchild), _p(t.child_begin), _p(t.pbegin), _p(t.pcount),
                          _p(mom32), _p(mac), C.c_int32(mac_kind), _p(t.box), _p(t.gbegin), _p(t.gcount), _p(t.gbox),
                          C.c_int64(sel.shape[0]), _p(sel), C.c_float(eps), _p(npc), _p(npp), _p(acc),
                          _p(lc), C.c_int64(t.ncells), _p(ll), C.c_int64(t.ncells))
    out = dict(npc=npc, npp=npp, accpot=acc, mom32=mom32, mac=mac)
    if want_lists:
        out["cells"] = lc[: int(npc[sel[0]])]
        out["leaves"] = ll[ll >= 0]
    return out


def direct(pos_mass, eps: float, t0: int = 0, t1: int | None = None):
    """O(N^2) binary64 direct sum for targets [t0, t1): float64[N,4] (NaN outside the range)."""
    pm = _f32c(pos_mass)
    n = pm.shape[0]
    t1 = n if t1 is None else t1
    acc = np.full((n, 4), np.nan, np.float64)
    lib().orc_direct(C.c_int64(n), _p(pm), C.c_float(eps), C.c_int64(t0), C.c_int64(t1), _p(acc))
    return acc


def kick(vel, acc, h):
    """O11 kick, in place on a float32[N,4] copy: v = fmaf(a, h, v)."""
    v = np.array(vel, dtype=np.float32, order="C", copy=True)
    a = np.ascontiguousarray(acc, np.float32)
    lib().orc_kick(C.c_int64(v.shape[0]), _p(v), _p(a), C.c_float(h))
    return v


def drift(pos_mass, vel, dt):
    """O11 drift: x = fmaf(v, dt, x)."""
    p = np.array(pos_mass, dtype=np.float32, order="C", copy=True)
    v = np.ascontiguousarray(vel, np.float32)
    lib().orc_drift(C.c_int64(p.shape[0]), _p(p), _p(v), C.c_float(dt))
    return p


@dataclass
class State:
    """Everything one force evaluation produces, in sorted (key) order."""
    pos: np.ndarray      # float32[N,4] sorted
    vel: np.ndarray      # float32[N,4] sorted
    ids: np.ndarray      # uint32[N]  caller identity of each sorted particle
    perm: np.ndarray     # uint32[N]  position in the INPUT arrays of each sorted particle
    keys: np.ndarray     # uint64[N]  sorted
    lo: np.ndarray
    e: int
    tree: Tree
    npc: np.ndarray = None
    npp: np.ndarray = None
    accpot: np.ndarray = None   # float64[N,4]
    mom32: np.ndarray = None
    mac: np.ndarray = None


def tree_build(pos_mass, vel=None, ids=None, nleaf: int = NLEAF, ncrit: int = NCRIT) -> State:
    """O1-O8 on unsorted inputs."""
    pm = _f32c(pos_mass)
    n = pm.shape[0]
    vel = np.zeros((n, 4), np.float32) if vel is None else _f32c(vel)
    ids = np.arange(n, dtype=np.uint32) if ids is None else np.ascontiguousarray(ids, np.uint32)
    lo, hi, e, ok = domain(pm)
    if not ok:
        raise ValueError("non-finite position or mass <= 0")
    k = keys(pm, lo, e)
    perm = sort_perm(k)
    ks = k[perm]
    ps, vs, idss = pm[perm], vel[perm], ids[perm]   # O5
    t = build_tree(ks, nleaf)
    make_groups(t, ncrit)
    moments(t, ps)
    return State(ps, vs, idss, perm, ks, lo, e, t)


def compute_forces(st: State, theta: float, eps: float, sel=None, forces: bool = True, mac_kind: int = MAC_EQ1) -> State:
    """O9 + O10."""
    r = walk_forces(st.tree, st.pos, theta, eps, sel=sel, forces=forces, mac_kind=mac_kind)
    st.npc, st.npp, st.accpot, st.mom32, st.mac = r["npc"], r["npp"], r["accpot"], r["mom32"], r["mac"]
    return st


def leapfrog_step(st: State, theta: float, eps: float, dt: float, nleaf: int = NLEAF, ncrit: int = NCRIT) -> State:
    """O11: kick(dt/2) with the held accelerations, drift(dt), O1-O10 on the new positions, kick(dt/2).

    The held accelerations are rounded to float32 (that is what an fp32 integrator holds).
    """
    h = np.float32(0.5) * np.float32(dt)
    a32 = st.accpot.astype(np.float32)
    v = kick(st.vel, a32, h)
    p = drift(st.pos, v, np.float32(dt))
    s2 = tree_build(p, v, st.ids, nleaf, ncrit)
    compute_forces(s2, theta, eps)
    s2.vel = kick(s2.vel, s2.accpot.astype(np.float32), h)
    return s2


# ---------------------------------------------------------------------------------------------- block time-steps (reading A29)
@dataclass
class BlockState:
    """Key-sorted particle state of the block time-step scheme: (pos, vel, accb) of particle i hold at tick[i]."""
    pos: np.ndarray      # float32[N,4]
    vel: np.ndarray      # float32[N,4]
    accb: np.ndarray     # float32[N,4]  held acceleration + potential (at the particle's own time)
    ids: np.ndarray      # uint32[N]
    tick: np.ndarray     # uint32[N]    time of the last update, in units of dt_max / 2^R
    rung: np.ndarray     # uint8[N]     dt_i = dt_max / 2^rung
    tree: Tree
    len_scale: float
    eta: float
    dt_max: float
    R: int
    now: int = 0         # system time in ticks
    active: np.ndarray = None
    npc: np.ndarray = None
    npp: np.ndarray = None


def rungs(acc, active, len_scale, eta, dt_max, R, tick, out=None):
    """A29 criterion: rung of the active particles (all if active is None) from their accelerations."""
    a = np.ascontiguousarray(acc, np.float32)
    n = a.shape[0]
    out = np.zeros(n, np.uint8) if out is None else out
    act = None if active is None else np.ascontiguousarray(active, np.uint8)
    lib().orc_rungs(C.c_int64(n), _p(a), _p(act), C.c_float(len_scale), C.c_float(eta), C.c_float(dt_max), C.c_int32(R),
                    C.c_uint32(tick), _p(out))
    return out


def block_init(st: State, len_scale: float, eta: float, dt_max: float, R: int) -> BlockState:
    """All particles synchronised at tick 0 with the forces of `st`; rungs from the criterion."""
    accb = np.ascontiguousarray(st.accpot, np.float64).astype(np.float32)
    r = rungs(accb, None, len_scale, eta, dt_max, R, 0)
    return BlockState(st.pos.copy(), st.vel.copy(), accb, st.ids.copy(), np.zeros(st.tree.n, np.uint32), r, st.tree,
                      float(len_scale), float(eta), float(dt_max), int(R))


def block_active(bs: BlockState):
    """(tick_next, active uint8[N])."""
    act = np.zeros(bs.tree.n, np.uint8)
    lib().orc_block_active.restype = C.c_uint32
    nxt = int(lib().orc_block_active(C.c_int64(bs.tree.n), _p(bs.tick), _p(bs.rung), C.c_int32(bs.R), _p(act)))
    return nxt, act


def block_step(bs: BlockState, theta: float, eps: float, acc_new=None) -> BlockState:
    """One system step on the EXISTING cells and groups: active set, predictor, moments (+ group boxes) of the moved
    particles, walk + forces of the groups with an active particle, corrector, new rungs.  acc_new (float32[N,4]): use
    these accelerations instead of the oracle's own (per-call parity: the integer decisions then follow the same floats)."""
    t = bs.tree
    nxt, act = block_active(bs)
    L = lib()
    L.orc_block_predict(C.c_int64(t.n), _p(bs.pos), _p(bs.vel), _p(bs.accb), _p(act), _p(bs.rung), C.c_float(bs.dt_max))
    moments(t, bs.pos)
    sel = np.nonzero(np.add.reduceat(act.astype(np.int64), t.gbegin) > 0)[0].astype(np.int64)
    r = walk_forces(t, bs.pos, theta, eps, sel=sel)
    bs.npc, bs.npp = r["npc"], r["npp"]
    new = np.nan_to_num(r["accpot"]).astype(np.float32) if acc_new is None else np.ascontiguousarray(acc_new, np.float32)
    bs.acc_eval = r["accpot"]
    L.orc_block_correct(C.c_int64(t.n), _p(bs.vel), _p(bs.accb), _p(new), _p(act), _p(bs.rung), C.c_float(bs.dt_max),
                        C.c_uint32(nxt), _p(bs.tick))
    rungs(bs.accb, act, bs.len_scale, bs.eta, bs.dt_max, bs.R, nxt, out=bs.rung)
    bs.now, bs.active = nxt, act
    return bs
