"""The acceleration-error experiment of PAPER.md:196-204 (section 4.2.1, Eq.2, Fig.8-9), on synthetic Plummer spheres.

    python -m paper_1106_1900_b200.accuracy [--n 32768 131072 1048576] [--theta 0.2 0.3 ... 0.8] [--eps 0.0] [--mac 0|1]

For every N: one tree build, one binary64 direct summation on the GPU (bh_direct_forces, the paper's "double precision
version of Sapporo"), then for every opening angle the fp32 tree forces (bh_compute_forces) and the distribution of
    da/a = |a_tree - a_direct| / |a_direct|                                  (Eq.2)
over all particles.  Printed per (N, theta), one JSON line: the error that 50 %, 10 % and 1 % of the particles exceed
(the three dotted lines of Fig.8; Fig.9 plots the first and the last against theta), the mean interaction counts and
the walk time.  Softening 0 as in the paper (L200).  The paper's own curves are images (A24): nothing is compared with
them; the claim that can be checked is "nearly independent of N" (L204).
Every force comes from the CUDA library; this module only draws inputs, marshals and takes percentiles on the host.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bh_inputs  # noqa: E402  (seeded input generators only; no method arithmetic)

from .binding import BarnesHut, direct_forces  # noqa: E402


def relative_error(a_tree: np.ndarray, a_direct: np.ndarray) -> np.ndarray:
    """Eq.2 per particle, in float64."""
    d = a_tree[:, :3].astype(np.float64) - a_direct[:, :3]
    return np.linalg.norm(d, axis=1) / np.linalg.norm(a_direct[:, :3], axis=1)


def exceeded_by(err: np.ndarray, fraction: float) -> float:
    """The error that `fraction` of the particles exceed (Fig.8: 0.5, 0.1, 0.01)."""
    return float(np.quantile(err, 1.0 - fraction))


def run(n: int, thetas, eps: float, seed: int | None = None, mac: int = 0):
    pm, vel, _ = bh_inputs.make("c2", n=n, seed=seed)
    bh = BarnesHut(n)
    bh.set_particles(pm, vel)
    bh.set_mac(mac)
    bh.tree_build()
    bh.compute_forces(float(thetas[0]), eps)
    t = bh.export_tree()                                   # sorted particles (device views of the workspace)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    ref = direct_forces(t["pos_mass"], eps)
    ev1.record()
    torch.cuda.synchronize()
    direct_ms = ev0.elapsed_time(ev1)
    a_direct = ref.cpu().numpy()
    out = []
    for th in thetas:
        ev0.record()
        bh.compute_forces(float(th), eps)
        ev1.record()
        st = bh.sync_status()
        walk_ms = ev0.elapsed_time(ev1)
        a_tree = t["acc_pot"].cpu().numpy()
        err = relative_error(a_tree, a_direct)
        out.append({"n": n, "theta": float(th), "eps": eps, "mac": "min_distance" if mac else "eq1", "exceeded_by_50pct": exceeded_by(err, 0.5),
                    "exceeded_by_10pct": exceeded_by(err, 0.1), "exceeded_by_1pct": exceeded_by(err, 0.01), "max": float(err.max()),
                    "pp_per_particle": st.sum_pp / n, "pc_per_particle": st.sum_pc / n, "walk_ms": walk_ms,
                    "direct_ms": direct_ms, "direct_pairs_per_s": n * (n - 1) / (direct_ms * 1e-3)})
    bh.close()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, nargs="+", default=[32768, 131072, 1048576])
    ap.add_argument("--theta", type=float, nargs="+", default=[0.2, 0.3, 0.4, 0.5, 0.6, 0.7, 0.8])
    ap.add_argument("--eps", type=float, default=0.0)
    ap.add_argument("--mac", type=int, default=0, choices=[0, 1], help="0: Eq.1; 1: minimum-distance MAC (PAPER.md:129)")
    args = ap.parse_args()
    for n in args.n:
        for row in run(n, args.theta, args.eps, mac=args.mac):
            print(json.dumps(row), flush=True)


if __name__ == "__main__":
    main()
