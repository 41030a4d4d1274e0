"""Toy outer-tracker geometry of BASELINE.json's configs (no method arithmetic).

PAPER.md:23 -- "each layer comprises of 2 closely-spaced silicon sensors"; a
*module* here is one (phi, z) tile (barrel) or (ring, phi) tile (endcap) of a
layer together with its two sensors.  Sensor ids are ``2*module + s`` with
``s = 0`` the lower sensor (smaller r in the barrel, smaller |z| in the
endcap) and ``s = 1`` the upper one.

Readings (G3/G4): ideal cylinders / planes; lower barrel sensor at
``r_layer``, upper at ``r_layer + 0.26`` cm; endcap lower at ``|z_disk|``, upper
at ``|z_disk| + 0.4`` cm; ``nphi = ceil(2*pi*r / 10 cm)`` equal tiles; endcap
disks cut into 9 equal rings over 23..110 cm.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BARREL_R = np.array([23.0, 36.0, 51.0, 68.0, 88.0, 108.0])
BARREL_GAP = 0.26
ENDCAP_Z = np.array([130.0, 160.0, 190.0, 225.0, 265.0])
ENDCAP_GAP = 0.4
ENDCAP_RMIN = 23.0
ENDCAP_RMAX = 110.0
ENDCAP_NRINGS = 9
TILE = 10.0

SUBDET_BARREL = 0
SUBDET_ENDCAP = 1


@dataclass
class Geometry:
    name: str
    barrel_zmax: float
    has_endcap: bool
    barrel_nphi: np.ndarray = field(default=None)
    barrel_nz: int = 0
    barrel_base: np.ndarray = field(default=None)
    endcap_nphi: np.ndarray = field(default=None)
    endcap_ring_edges: np.ndarray = field(default=None)
    endcap_base: np.ndarray = field(default=None)  # [side(0:-z,1:+z), disk, ring]
    n_modules: int = 0
    # per-module table (what lst_load_geometry receives)
    subdet: np.ndarray = field(default=None)
    layer: np.ndarray = field(default=None)
    side: np.ndarray = field(default=None)
    ring: np.ndarray = field(default=None)

    # ---- volume limits used by the event generator -------------------------
    @property
    def r_exit(self) -> float:
        return 112.0

    @property
    def z_exit(self) -> float:
        return float(ENDCAP_Z[-1] + 5.0) if self.has_endcap else self.barrel_zmax

    @property
    def n_sensors(self) -> int:
        return 2 * self.n_modules

    # ---- surface lists -----------------------------------------------------
    def barrel_surfaces(self):
        """(radius, layer index 0..5, sensor 0/1) for the 12 barrel cylinders."""
        out = []
        for il, r in enumerate(BARREL_R):
            out.append((float(r), il, 0))
            out.append((float(r + BARREL_GAP), il, 1))
        return out

    def endcap_surfaces(self):
        """(z, side index 0/1, disk index 0..4, sensor 0/1) for the 20 endcap planes."""
        out = []
        if not self.has_endcap:
            return out
        for iside, sgn in enumerate((-1.0, 1.0)):
            for idisk, z in enumerate(ENDCAP_Z):
                out.append((float(sgn * z), iside, idisk, 0))
                out.append((float(sgn * (z + ENDCAP_GAP)), iside, idisk, 1))
        return out

    # ---- position -> module -----------------------------------------------
    def barrel_module(self, il, phi, z):
        """Module index of barrel layer ``il`` (0..5) at azimuth ``phi`` and ``z``."""
        il = np.asarray(il)
        nphi = self.barrel_nphi[il]
        p = np.mod(phi, 2.0 * np.pi)
        iphi = np.minimum((p / (2.0 * np.pi) * nphi).astype(np.int64), nphi - 1)
        iz = np.floor((np.asarray(z) + self.barrel_zmax) / TILE).astype(np.int64)
        iz = np.clip(iz, 0, self.barrel_nz - 1)
        return (self.barrel_base[il] + iz * nphi + iphi).astype(np.int64)

    def endcap_module(self, iside, idisk, r, phi):
        r = np.asarray(r)
        w = (ENDCAP_RMAX - ENDCAP_RMIN) / ENDCAP_NRINGS
        ir = np.clip(np.floor((r - ENDCAP_RMIN) / w).astype(np.int64), 0, ENDCAP_NRINGS - 1)
        nphi = self.endcap_nphi[ir]
        p = np.mod(phi, 2.0 * np.pi)
        iphi = np.minimum((p / (2.0 * np.pi) * nphi).astype(np.int64), nphi - 1)
        return (self.endcap_base[np.asarray(iside), np.asarray(idisk), ir] + iphi).astype(np.int64)

    def module_table(self) -> np.ndarray:
        """int32 [n_modules, 4] = (subdet, layer, side, ring) -- the lst_module records."""
        return np.stack([self.subdet, self.layer, self.side, self.ring], axis=1).astype(np.int32)


def make_geometry(name: str) -> Geometry:
    """``barrel_z60`` (configs 1, 2, 4) or ``barrel_z120_endcap`` (configs 3, 5)."""
    if name == "barrel_z60":
        g = Geometry(name=name, barrel_zmax=60.0, has_endcap=False)
    elif name == "barrel_z120_endcap":
        g = Geometry(name=name, barrel_zmax=120.0, has_endcap=True)
    else:
        raise ValueError(f"unknown geometry {name!r}")

    g.barrel_nphi = np.ceil(2.0 * np.pi * BARREL_R / TILE).astype(np.int64)
    g.barrel_nz = int(round(2.0 * g.barrel_zmax / TILE))
    per_layer = g.barrel_nphi * g.barrel_nz
    g.barrel_base = np.concatenate([[0], np.cumsum(per_layer)[:-1]]).astype(np.int64)
    n = int(per_layer.sum())

    subdet = [np.full(n, SUBDET_BARREL)]
    layer = [np.repeat(np.arange(1, 7), per_layer)]
    side = [np.zeros(n, dtype=np.int64)]
    ring = [np.concatenate([np.repeat(np.arange(g.barrel_nz), g.barrel_nphi[il]) for il in range(6)])]

    if g.has_endcap:
        edges = np.linspace(ENDCAP_RMIN, ENDCAP_RMAX, ENDCAP_NRINGS + 1)
        g.endcap_ring_edges = edges
        rmid = 0.5 * (edges[:-1] + edges[1:])
        g.endcap_nphi = np.ceil(2.0 * np.pi * rmid / TILE).astype(np.int64)
        g.endcap_base = np.zeros((2, len(ENDCAP_Z), ENDCAP_NRINGS), dtype=np.int64)
        for iside in range(2):
            for idisk in range(len(ENDCAP_Z)):
                for ir in range(ENDCAP_NRINGS):
                    g.endcap_base[iside, idisk, ir] = n
                    k = int(g.endcap_nphi[ir])
                    subdet.append(np.full(k, SUBDET_ENDCAP))
                    layer.append(np.full(k, idisk + 1))
                    side.append(np.full(k, -1 if iside == 0 else 1))
                    ring.append(np.full(k, ir))
                    n += k
    else:
        g.endcap_nphi = np.zeros(0, dtype=np.int64)
        g.endcap_base = np.zeros((2, 0, 0), dtype=np.int64)

    g.n_modules = n
    g.subdet = np.concatenate(subdet).astype(np.int32)
    g.layer = np.concatenate(layer).astype(np.int32)
    g.side = np.concatenate(side).astype(np.int32)
    g.ring = np.concatenate(ring).astype(np.int32)
    assert g.subdet.shape[0] == n
    return g
