"""Module connection map, precomputed on the host (reading S4).

Edges m -> m' where m' is the NEXT module crossed (lower-sensor surfaces, in
path order) by a pT >= 0.8 GeV helix leaving the beam line at |z0| <= 15 cm.
Built by a seeded Monte-Carlo scan over (phi, eta, z0, signed 1/pT); the map
is an INPUT of the method: oracle and CUDA path read the same CSR arrays.
No skip-layer edges by default; ``skip=True`` adds the edges
m -> m'' to the module crossed AFTER the next one, so that a Line Segment can bridge a layer
that has no hit.  The scan is cached under ``lst_inputs/_cache`` (a pure
speed-up: the same seed regenerates the same map).
"""
from __future__ import annotations

import os

import numpy as np

from .geometry import BARREL_R, ENDCAP_RMAX, ENDCAP_RMIN, ENDCAP_Z, Geometry
from .helix import Tracks

PT_MIN_MAP = 0.8
Z0_MAX_MAP = 15.0
_CACHE_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "_cache")
_CACHE_VERSION = 2


def _scan_chunk(geom: Geometry, rng: np.random.Generator, n: int, eta_max: float, skip: bool = False):
    phi0 = rng.uniform(0.0, 2.0 * np.pi, n)
    eta = rng.uniform(-eta_max, eta_max, n)
    z0 = rng.uniform(-Z0_MAX_MAP, Z0_MAX_MAP, n)
    inv_pt = rng.uniform(-1.0 / PT_MIN_MAP, 1.0 / PT_MIN_MAP, n)
    inv_pt = np.where(np.abs(inv_pt) < 1e-3, 1e-3, inv_pt)
    trk = Tracks(np.zeros(n), np.zeros(n), z0, phi0, eta, 1.0 / np.abs(inv_pt), np.sign(inv_pt))
    t_exit = trk.t_exit(geom.r_exit, geom.z_exit, np.pi)  # outgoing half turn only

    ts, mods = [], []
    for il, r in enumerate(BARREL_R):
        t = trk.cyl_crossings(float(r), 1).min(axis=1)  # first (outgoing) crossing
        x, y, z = trk.pos(t)
        ok = np.isfinite(t) & (t < t_exit) & (np.abs(z) < geom.barrel_zmax)
        m = geom.barrel_module(np.full(n, il), np.arctan2(y, x), np.where(ok, z, 0.0))
        ts.append(np.where(ok, t, np.inf))
        mods.append(np.where(ok, m, -1))
    if geom.has_endcap:
        for iside, sgn in enumerate((-1.0, 1.0)):
            for idisk, zd in enumerate(ENDCAP_Z):
                t = trk.plane_crossing(float(sgn * zd))
                x, y, _ = trk.pos(np.where(np.isfinite(t), t, 0.0))
                r = np.hypot(x, y)
                ok = np.isfinite(t) & (t < t_exit) & (r >= ENDCAP_RMIN) & (r < ENDCAP_RMAX)
                m = geom.endcap_module(
                    np.full(n, iside), np.full(n, idisk), np.where(ok, r, ENDCAP_RMIN), np.arctan2(y, x)
                )
                ts.append(np.where(ok, t, np.inf))
                mods.append(np.where(ok, m, -1))
    ts = np.stack(ts, axis=1)
    mods = np.stack(mods, axis=1)
    order = np.argsort(ts, axis=1, kind="stable")
    mods = np.take_along_axis(mods, order, axis=1)
    a = mods[:, :-1].ravel()
    b = mods[:, 1:].ravel()
    if skip:  # also the crossing after the next one (invalid crossings sort last: t = inf)
        a = np.concatenate([a, mods[:, :-2].ravel()])
        b = np.concatenate([b, mods[:, 2:].ravel()])
    keep = (a >= 0) & (b >= 0)
    return a[keep], b[keep]


def build_connection_map(geom: Geometry, n_samples: int | None = None, seed: int = 12345, cache: bool = True,
                         skip: bool = False):
    """Return CSR ``(offsets int32[n_modules+1], targets int32[n_edges])``, targets sorted per row."""
    if n_samples is None:
        n_samples = 3_000_000 if geom.has_endcap else 1_000_000
    tag = f"{geom.name}_n{n_samples}_s{seed}_v{_CACHE_VERSION}{'_skip' if skip else ''}.npz"
    path = os.path.join(_CACHE_DIR, tag)
    if cache and os.path.exists(path):
        with np.load(path) as f:
            return f["offsets"], f["targets"]

    eta_max = float(np.arcsinh(geom.z_exit / BARREL_R[0])) + 0.1
    rng = np.random.Generator(np.random.PCG64(seed))
    nm = geom.n_modules
    keys = np.zeros(0, dtype=np.int64)
    chunk = 250_000
    done = 0
    while done < n_samples:
        n = min(chunk, n_samples - done)
        a, b = _scan_chunk(geom, rng, n, eta_max, skip)
        keys = np.union1d(keys, np.unique(a.astype(np.int64) * nm + b.astype(np.int64)))
        done += n
    src = (keys // nm).astype(np.int64)
    dst = (keys % nm).astype(np.int32)
    counts = np.bincount(src, minlength=nm)
    offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    targets = dst  # keys are sorted => grouped by src, ascending dst
    if cache:
        try:
            os.makedirs(_CACHE_DIR, exist_ok=True)
            tmp = path + f".tmp{os.getpid()}.npz"
            np.savez(tmp, offsets=offsets, targets=targets)
            os.replace(tmp, path)
        except OSError:
            pass
    return offsets, targets
