"""Shared helpers of the GPU parity tests: run the CUDA path through the C ABI, run the oracle, compare.

Bit-exact: keys, perm, topology, groups, fp64 moments, boxes, fp32 roundings, opening radii, per-group counts.
Tolerance (BASELINE.json north_star): accelerations and potentials, relative error RMS <= 1e-5 and max <= 1e-4
against the oracle's binary64 evaluation of the same interaction lists.
"""
from __future__ import annotations

import numpy as np

import oracle

RMS_TOL = 1e-5
MAX_TOL = 1e-4


def gpu_tree(bh, pos_mass, vel, theta, eps, ids=None, mac=0):
    """set_particles + tree_build + compute_forces + export, as numpy arrays."""
    bh.set_particles(pos_mass, vel, ids)
    bh.set_mac(mac)
    bh.tree_build()
    bh.compute_forces(theta, eps)
    return export_numpy(bh)


def export_numpy(bh):
    t = bh.export_tree()
    out = {}
    for k, v in t.items():
        out[k] = v.cpu().numpy() if hasattr(v, "cpu") else v
    out["key"] = out["key"].astype(np.uint64)
    out["cell_prefix"] = out["cell_prefix"].astype(np.uint64)
    return out


def compare_tree(g, st, problems=None, check_vel=True):
    """Bit-exact comparison of everything but the forces.  Returns the list of mismatching items."""
    bad = [] if problems is None else problems
    t = st.tree

    def eq(name, a, b):
        a, b = np.asarray(a), np.asarray(b)
        if a.shape != b.shape:
            bad.append(f"{name}: shape {a.shape} vs {b.shape}")
        elif not np.array_equal(a, b):
            w = np.argwhere(a != b)
            bad.append(f"{name}: {w.shape[0]} of {a.size} differ, first at {tuple(w[0])}: gpu {a[tuple(w[0])]} oracle {b[tuple(w[0])]}")

    s = g["stats"]
    eq("domain lo", np.array(list(s.lo), np.float32), st.lo)
    eq("domain exp", s.domain_exp, st.e)
    eq("keys", g["key"], st.keys)
    eq("perm", g["perm"].astype(np.int64), st.perm.astype(np.int64))
    eq("ids", g["id"].astype(np.int64), st.ids.astype(np.int64))
    eq("pos sorted", g["pos_mass"], st.pos)
    if check_vel:
        eq("vel sorted", g["vel"], st.vel)
    eq("n_cells", g["n_cells"], t.ncells)
    eq("n_groups", g["n_groups"], t.ngroups)
    if g["n_cells"] != t.ncells or g["n_groups"] != t.ngroups:
        return bad
    eq("level_offset", g["level_offset"].astype(np.int64), t.level_offset)
    eq("cell_level", g["cell_level"], t.level)
    eq("cell_prefix", g["cell_prefix"], t.prefix)
    eq("cell_pbegin", g["cell_pbegin"].astype(np.int64), t.pbegin)
    eq("cell_pcount", g["cell_pcount"].astype(np.int64), t.pcount)
    eq("cell_child_begin", g["cell_child_begin"].astype(np.int64), t.child_begin)
    eq("cell_nchild", g["cell_nchild"], t.nchild)
    eq("cell_parent", g["cell_parent"].astype(np.int64), t.parent)
    eq("group_begin", g["group_begin"][:-1].astype(np.int64), t.gbegin)
    eq("group_end", g["group_begin"][-1], t.n)
    eq("group_cell", g["group_cell"].astype(np.int64), t.gcell)
    eq("cell_mom64", g["cell_mom64"].view(np.uint64), t.mom64.view(np.uint64))
    eq("cell_box", g["cell_box"].view(np.uint32), t.box.view(np.uint32))
    if st.mom32 is not None:
        eq("cell_mom32", g["cell_mom32"].view(np.uint32), st.mom32.view(np.uint32))
        eq("cell_r2open", g["cell_r2open"].view(np.uint32), np.ascontiguousarray(st.mac[:, 2]).view(np.uint32))
        # the records the walk kernels really read (not a re-export): MAC record and evaluation record, from the oracle's fp32 moments
        m = st.mom32
        f = np.float32
        T = ((m[:, 4] + m[:, 5]).astype(f) + m[:, 6]).astype(f)
        trec = np.column_stack([m[:, 1], m[:, 2], m[:, 3], st.mac[:, 2]]).astype(f)
        erec = np.column_stack([m[:, 1], m[:, 2], m[:, 3], m[:, 0], f(-3) * m[:, 4], f(-3) * m[:, 5], f(-3) * m[:, 6], f(-3) * m[:, 7],
                                f(-3) * m[:, 8], f(-3) * m[:, 9], f(-0.5) * T, f(-1.5) * T]).astype(f)
        eq("cell_trec", g["cell_trec"].view(np.uint32), np.ascontiguousarray(trec).view(np.uint32))
        eq("cell_erec", g["cell_erec"].view(np.uint32), np.ascontiguousarray(erec).view(np.uint32))
    return bad


def compare_counts(g, st, sel=None, problems=None):
    bad = [] if problems is None else problems
    sel = np.arange(st.tree.ngroups) if sel is None else np.asarray(sel)
    for name, a, b in (("n_pc", g["group_npc"], st.npc), ("n_pp", g["group_npp"], st.npp)):
        a, b = a[sel].astype(np.int64), b[sel]
        if not np.array_equal(a, b):
            w = np.nonzero(a != b)[0]
            bad.append(f"{name}: {w.size} of {a.size} groups differ, first group {sel[w[0]]}: gpu {a[w[0]]} oracle {b[w[0]]}")
    return bad


def force_errors(g, st, sel=None):
    """Relative errors of acceleration and potential over the particles of the selected groups."""
    t = st.tree
    if sel is None:
        idx = np.arange(t.n)
    else:
        idx = np.concatenate([np.arange(t.gbegin[k], t.gbegin[k] + t.gcount[k]) for k in sel])
    a = g["acc_pot"][idx].astype(np.float64)
    r = st.accpot[idx]
    ea = np.linalg.norm(a[:, :3] - r[:, :3], axis=1) / np.linalg.norm(r[:, :3], axis=1)
    ep = np.abs(a[:, 3] - r[:, 3]) / np.abs(r[:, 3])
    return dict(acc_rms=float(np.sqrt(np.mean(ea ** 2))), acc_max=float(ea.max()),
                pot_rms=float(np.sqrt(np.mean(ep ** 2))), pot_max=float(ep.max()), n=int(idx.size))


def check_forces(g, st, sel=None):
    e = force_errors(g, st, sel)
    assert e["acc_rms"] <= RMS_TOL and e["acc_max"] <= MAX_TOL, e
    assert e["pot_rms"] <= RMS_TOL and e["pot_max"] <= MAX_TOL, e
    return e


def oracle_state(pos_mass, vel, theta, eps, ids=None, sel=None, forces=True, nleaf=16, ncrit=64, mac=0):
    st = oracle.tree_build(pos_mass, vel, ids, nleaf, ncrit)
    oracle.compute_forces(st, theta, eps, sel=sel, forces=forces, mac_kind=mac)
    return st
