"""Vortex tracking on the CUDA path (Figs. 18, 21, 22: the
paper follows "vortices with a positive / negative winding number" of each m_f as red / blue tracks).

The device does the work -- `qlga_vortices` (plaquette winding numbers) and `qlga_vortex_match` (mutual
nearest neighbours of equal channel and winding under the periodic metric, an O(n m) search) -- and this
module keeps the books: track identities, births, deaths, unwrapped positions (reading R18).

    tr = VortexTracker(sim, max_dist=6)
    for _ in range(n): sim.step(k); tr.update()
    tr.tracks[id] -> Track(j, w, steps[], x[], y[])      # x, y unwrapped: they leave [0, N) as the vortex drifts
"""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass
class Track:
    ident: int
    j: int                 # channel, m_f = 2 - j
    w: int                 # winding number of the plaquette, +1 or -1
    steps: list
    x: list                # plaquette coordinates, unwrapped (continuous across the periodic boundary)
    y: list
    alive: bool = True

    def displacement(self):
        return self.x[-1] - self.x[0], self.y[-1] - self.y[0]


def canonical(records):
    """records sorted by (j, y, x): the detector's output order is unspecified."""
    r = np.asarray(records, dtype=np.int32).reshape(-1, 4)
    return r[np.lexsort((r[:, 1], r[:, 2], r[:, 0]))]


class VortexTracker:
    def __init__(self, sim, max_dist=8, max_vortices=65536):
        assert sim.ndim == 2
        self.sim, self.max_dist2, self.max_vortices = sim, int(max_dist) ** 2, int(max_vortices)
        self.tracks = {}
        self.events = []           # (step, "birth" | "death", ident)
        self._prev = None          # canonical records of the last detection
        self._ids = None           # track id of every record of the last detection
        self._next = 0

    def update(self):
        """Detect on the current state, associate with the previous detection; returns the canonical records
        and the track id of each."""
        step = self.sim.observables()["step"]
        rec, count = self.sim.vortices(self.max_vortices)
        if count > self.max_vortices:
            raise RuntimeError(f"{count} vortices: more than max_vortices = {self.max_vortices}")
        cur = canonical(rec)
        ids = np.full(len(cur), -1, dtype=np.int64)
        if self._prev is not None:
            mc, mp = self.sim.vortex_match(self._prev, cur, self.max_dist2)
            for k in np.nonzero(mp < 0)[0]:
                t = self.tracks[int(self._ids[k])]
                t.alive = False
                self.events.append((step, "death", t.ident))
            for i in np.nonzero(mc >= 0)[0]:
                t = self.tracks[int(self._ids[mc[i]])]
                ids[i] = t.ident
                # minimal-image displacement from the last recorded plaquette
                px, py = self._prev[mc[i], 1], self._prev[mc[i], 2]
                dx = (int(cur[i, 1]) - int(px) + self.sim.nx // 2) % self.sim.nx - self.sim.nx // 2
                dy = (int(cur[i, 2]) - int(py) + self.sim.ny // 2) % self.sim.ny - self.sim.ny // 2
                t.steps.append(step); t.x.append(t.x[-1] + dx); t.y.append(t.y[-1] + dy)
        for i in np.nonzero(ids < 0)[0]:
            t = Track(self._next, int(cur[i, 0]), int(cur[i, 3]), [step], [int(cur[i, 1])], [int(cur[i, 2])])
            self.tracks[t.ident] = t
            ids[i] = t.ident
            self._next += 1
            if self._prev is not None:
                self.events.append((step, "birth", t.ident))
        self._prev, self._ids = cur, ids
        return cur, ids

    def total_winding(self):
        """Sum of the windings of the live tracks, per channel (conserved: 0 on a periodic lattice)."""
        tot = np.zeros(5, dtype=np.int64)
        for t in self.tracks.values():
            if t.alive:
                tot[t.j] += t.w
        return tot
