"""Host-resident callers: independent force steps from pinned host buffers, two in flight.

A caller that holds its particles in host memory pays, per step, the upload of positions, velocities and ids and the
read-back of positions, velocities and accelerations (36 + 52 bytes per particle): at 1 M particles that is 1.7 ms of PCIe
time beside 2.6 ms of kernels.  PCIe is full duplex and the copy engines run beside the SMs, so two contexts on two
streams hide the copies of one step behind the kernels of the other.  This class is argument marshalling only: every
step is bh_set_particles + bh_tree_build + bh_compute_forces + bh_kick_drift + bh_get_particles on a BarnesHut
context (include/bh.h), exactly what a single-context caller would issue.
"""
from __future__ import annotations

import torch

from .binding import BarnesHut


class HostStepPipeline:
    """submit(pos_mass, vel, ids) enqueues one step (S0-S8 and the kick-drift of S9) on the next of `depth` contexts and
    returns a ticket; result(ticket) waits for that step and returns its pinned host buffers (pos_mass, vel, acc_pot, ids),
    valid until the same context is used again, i.e. for the next depth - 1 submissions."""

    def __init__(self, n: int, theta: float, eps: float, dt: float, depth: int = 2, device=None, mac: int = 0, **cfg):
        if depth < 1:
            raise ValueError("depth must be >= 1")
        self.n, self.theta, self.eps, self.dt, self.depth = int(n), float(theta), float(eps), float(dt), int(depth)
        self.ctx = [BarnesHut(n, device=device, **cfg) for _ in range(depth)]
        for c in self.ctx:
            c.set_mac(mac)
        dev = self.ctx[0].device
        self.streams = [torch.cuda.Stream(device=dev) for _ in range(depth)]
        self.out = [(torch.empty((n, 4), dtype=torch.float32).pin_memory(), torch.empty((n, 4), dtype=torch.float32).pin_memory(),
                     torch.empty((n, 4), dtype=torch.float32).pin_memory(), torch.empty(n, dtype=torch.int32).pin_memory())
                    for _ in range(depth)]
        self.submitted = 0

    def submit(self, pos_mass, vel, ids=None) -> int:
        """pos_mass, vel: pinned float32[n, 4]; ids: pinned int32 / uint32[n] or None.  The buffers must stay untouched until
        result() of this ticket (or of a later one on the same context) has returned."""
        k = self.submitted % self.depth
        s = self.streams[k]
        s.synchronize()                          # the step this context ran `depth` submissions ago has landed
        with torch.cuda.stream(s):
            c = self.ctx[k]
            c.set_particles(pos_mass, vel, ids)
            c.tree_build()
            c.compute_forces(self.theta, self.eps)
            c.kick_drift(self.dt, self.dt)
            c.get_particles(*self.out[k])
        t = self.submitted
        self.submitted += 1
        return t

    def result(self, ticket: int):
        if not (self.submitted - self.depth <= ticket < self.submitted):
            raise ValueError("the buffers of that ticket have been reused (or it was never submitted)")
        k = ticket % self.depth
        self.streams[k].synchronize()
        return self.out[k]

    def drain(self):
        for s in self.streams:
            s.synchronize()

    def close(self):
        self.drain()
        for c in self.ctx:
            c.close()
        self.ctx = []
