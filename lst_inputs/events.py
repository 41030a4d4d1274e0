"""Seeded synthetic events: outer-tracker hits and inner-tracker seeds (pLS).

Makes inputs only (float64 helix propagation, then cast to float32); holds no
selection arithmetic.  Recipe and readings G1..G7/S6 are listed in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .geometry import (
    BARREL_GAP,
    BARREL_R,
    ENDCAP_GAP,
    ENDCAP_NRINGS,
    ENDCAP_RMAX,
    ENDCAP_RMIN,
    ENDCAP_Z,
    TILE,
    Geometry,
)
from .helix import TWO_PI, Tracks

SIGMA_RPHI = 0.0030  # 30 um
SIGMA_Z = 0.15  # 1.5 mm (barrel: along z; endcap: along r)
PIXEL_R = (3.0, 7.0)
SIGMA_PIXEL = 0.0010  # 10 um

PLS_FIELDS = ("pt", "eta", "phi", "vx", "vy", "vz", "x0", "y0", "z0", "x1", "y1", "z1")


@dataclass
class EventSpec:
    n_tracks: int
    pt_dist: tuple  # ("loguniform", lo, hi) | ("power3", lo)
    eta_max: float
    max_turns: float = 2.0
    noise: tuple | None = None  # ("count", n) | ("frac", f)
    inefficiency: float = 0.0
    seeds: bool = False
    fake_seed_frac: float = 0.10
    n_displaced: int = 0
    d0_max: float = 20.0
    sigma_vz: float = 5.0
    phi_range: tuple = (0.0, TWO_PI)  # azimuth window of the generated helices
    # strip-like sensors (Fig. 1): on the barrel layers listed here (1-based) a hit's
    # z is the centre of its strip of length strip_pitch; on endcap rings starting at r >= strip_endcap_rmin
    # its r is the centre of one of the two strip rows of the ring.  0 = the default pixel-like sensors.
    strip_pitch: float = 0.0
    strip_layers: tuple = (4, 5, 6)
    strip_endcap_rmin: float = 60.0


@dataclass
class Event:
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    sensor: np.ndarray
    truth: np.ndarray  # generating track per hit, -1 = noise
    trk: dict = field(default_factory=dict)  # truth track parameters
    pls: dict = field(default_factory=dict)  # pLS SoA (float32) + "q" int32 + "truth" int32

    @property
    def n_hits(self) -> int:
        return int(self.x.shape[0])

    @property
    def n_pls(self) -> int:
        return int(self.pls["pt"].shape[0]) if self.pls else 0


def _sample_pt(rng, dist, n):
    if dist[0] == "loguniform":
        lo, hi = dist[1], dist[2]
        return np.exp(rng.uniform(np.log(lo), np.log(hi), n))
    if dist[0] == "power3":  # dN/dpT ~ pT^-3 above lo
        lo = dist[1]
        u = rng.uniform(0.0, 1.0, n)
        return np.minimum(lo / np.sqrt(1.0 - u), 200.0)
    raise ValueError(dist)


def _make_tracks(rng, spec: EventSpec):
    n = spec.n_tracks
    pt = _sample_pt(rng, spec.pt_dist, n)
    eta = rng.uniform(-spec.eta_max, spec.eta_max, n)
    phi0 = rng.uniform(spec.phi_range[0], spec.phi_range[1], n)
    z0 = rng.normal(0.0, spec.sigma_vz, n)
    q = np.where(rng.uniform(size=n) < 0.5, -1.0, 1.0)
    d0 = np.zeros(n)
    if spec.n_displaced:
        k = spec.n_displaced
        pt = np.concatenate([pt, _sample_pt(rng, spec.pt_dist, k)])
        eta = np.concatenate([eta, rng.uniform(-spec.eta_max, spec.eta_max, k)])
        phi0 = np.concatenate([phi0, rng.uniform(spec.phi_range[0], spec.phi_range[1], k)])
        z0 = np.concatenate([z0, rng.normal(0.0, spec.sigma_vz, k)])
        q = np.concatenate([q, np.where(rng.uniform(size=k) < 0.5, -1.0, 1.0)])
        d0 = np.concatenate([d0, rng.uniform(0.0, spec.d0_max, k)])
    # perigee point: transverse distance d0 from the beam line, perpendicular to the direction
    xs = d0 * np.sin(phi0)
    ys = -d0 * np.cos(phi0)
    return Tracks(xs, ys, z0, phi0, eta, pt, q), d0


def _strip_z(z, pitch):
    """Centre of the strip (length ``pitch``, edges at multiples of it) that holds z."""
    return (np.floor(z / pitch) + 0.5) * pitch


def _strip_r(r):
    """Centre of the strip row of an endcap ring that holds r (two rows per ring)."""
    w = (ENDCAP_RMAX - ENDCAP_RMIN) / ENDCAP_NRINGS
    ir = np.clip(np.floor((r - ENDCAP_RMIN) / w), 0, ENDCAP_NRINGS - 1)
    r1 = ENDCAP_RMIN + ir * w
    half = 0.5 * w
    row = np.clip(np.floor((r - r1) / half), 0, 1)
    return r1 + (row + 0.5) * half, r1


def _signal_hits(rng, geom: Geometry, trk: Tracks, spec: EventSpec):
    n = len(trk)
    n_turns = int(np.ceil(spec.max_turns))
    t_exit = trk.t_exit(geom.r_exit, geom.z_exit, spec.max_turns * TWO_PI)
    xs, ys, zs, sens, truth = [], [], [], [], []
    tid = np.arange(n)

    for rho, il, s in geom.barrel_surfaces():
        t = trk.cyl_crossings(rho, n_turns)  # [n, 2*n_turns]
        x, y, z = trk.pos(np.where(np.isfinite(t), t, 0.0))
        ok = np.isfinite(t) & (t < t_exit[:, None]) & (np.abs(z) < geom.barrel_zmax)
        ii, jj = np.nonzero(ok)
        if ii.size == 0:
            continue
        phi = np.arctan2(y[ii, jj], x[ii, jj]) + rng.normal(0.0, SIGMA_RPHI, ii.size) / rho
        zz = z[ii, jj] + rng.normal(0.0, SIGMA_Z, ii.size)
        if spec.strip_pitch > 0.0 and (il + 1) in spec.strip_layers:
            zz = _strip_z(zz, spec.strip_pitch)
        m = geom.barrel_module(np.full(ii.size, il), phi, zz)
        xs.append(rho * np.cos(phi))
        ys.append(rho * np.sin(phi))
        zs.append(zz)
        sens.append(2 * m + s)
        truth.append(tid[ii])

    for zd, iside, idisk, s in geom.endcap_surfaces():
        t = trk.plane_crossing(zd)
        x, y, _ = trk.pos(np.where(np.isfinite(t), t, 0.0))
        r = np.hypot(x, y)
        ok = np.isfinite(t) & (t < t_exit) & (r >= ENDCAP_RMIN) & (r < ENDCAP_RMAX)
        ii = np.nonzero(ok)[0]
        if ii.size == 0:
            continue
        rr = r[ii] + rng.normal(0.0, SIGMA_Z, ii.size)
        if spec.strip_pitch > 0.0:
            rq, r1 = _strip_r(rr)
            rr = np.where(r1 >= spec.strip_endcap_rmin, rq, rr)
        phi = np.arctan2(y[ii], x[ii]) + rng.normal(0.0, SIGMA_RPHI, ii.size) / r[ii]
        m = geom.endcap_module(np.full(ii.size, iside), np.full(ii.size, idisk), rr, phi)
        xs.append(rr * np.cos(phi))
        ys.append(rr * np.sin(phi))
        zs.append(np.full(ii.size, zd))
        sens.append(2 * m + s)
        truth.append(tid[ii])

    if not xs:
        e = np.zeros(0)
        return e, e, e, np.zeros(0, dtype=np.int64), np.zeros(0, dtype=np.int64)
    return (np.concatenate(xs), np.concatenate(ys), np.concatenate(zs),
            np.concatenate(sens).astype(np.int64), np.concatenate(truth).astype(np.int64))


def _noise_hits(rng, geom: Geometry, n: int, spec: EventSpec | None = None):
    """``n`` hits, each on a uniformly chosen sensor, uniform over that sensor's area (strip sensors: on a strip centre)."""
    sensor = rng.integers(0, geom.n_sensors, n)
    m = sensor // 2
    s = sensor % 2
    x = np.zeros(n)
    y = np.zeros(n)
    z = np.zeros(n)
    u1 = rng.uniform(size=n)
    u2 = rng.uniform(size=n)
    bar = geom.subdet[m] == 0
    if bar.any():
        mb = m[bar]
        il = geom.layer[mb] - 1
        loc = mb - geom.barrel_base[il]
        nphi = geom.barrel_nphi[il]
        iz = loc // nphi
        iphi = loc % nphi
        rho = BARREL_R[il] + s[bar] * BARREL_GAP
        phi = (iphi + u1[bar]) / nphi * TWO_PI
        x[bar] = rho * np.cos(phi)
        y[bar] = rho * np.sin(phi)
        zb = -geom.barrel_zmax + (iz + u2[bar]) * TILE
        if spec is not None and spec.strip_pitch > 0.0:
            zb = np.where(np.isin(il + 1, spec.strip_layers), _strip_z(zb, spec.strip_pitch), zb)
        z[bar] = zb
    end = ~bar
    if end.any():
        me = m[end]
        ir = geom.ring[me]
        idisk = geom.layer[me] - 1
        iside = (geom.side[me] > 0).astype(np.int64)
        iphi = me - geom.endcap_base[iside, idisk, ir]
        nphi = geom.endcap_nphi[ir]
        w = (ENDCAP_RMAX - ENDCAP_RMIN) / ENDCAP_NRINGS
        r1 = ENDCAP_RMIN + ir * w
        r2 = r1 + w
        r = np.sqrt(r1 * r1 + u2[end] * (r2 * r2 - r1 * r1))
        if spec is not None and spec.strip_pitch > 0.0:
            r = np.where(r1 >= spec.strip_endcap_rmin, _strip_r(r)[0], r)
        phi = (iphi + u1[end]) / nphi * TWO_PI
        x[end] = r * np.cos(phi)
        y[end] = r * np.sin(phi)
        z[end] = geom.side[me] * (ENDCAP_Z[idisk] + s[end] * ENDCAP_GAP)
    return x, y, z, sensor.astype(np.int64)


def _make_seeds(rng, trk: Tracks, d0, spec: EventSpec):
    """One pLS per track with pT > 0.8, |eta| < 4 that crosses both pixel radii, plus fakes."""
    n = len(trk)
    t0 = trk.cyl_crossings(PIXEL_R[0], 1).min(axis=1)
    t1 = trk.cyl_crossings(PIXEL_R[1], 1).min(axis=1)
    ok = (trk.pt > 0.8) & (np.abs(trk.eta) < 4.0) & np.isfinite(t0) & np.isfinite(t1) & (t0 < 1.0) & (t1 < 1.0) & (t0 < t1)
    idx = np.nonzero(ok)[0]
    n_fake = int(round(spec.fake_seed_frac * idx.size))
    if n_fake:
        fpt = _sample_pt(rng, ("loguniform", 0.8, 20.0), n_fake)
        fk = Tracks(np.zeros(n_fake), np.zeros(n_fake), rng.normal(0.0, spec.sigma_vz, n_fake),
                    rng.uniform(0.0, TWO_PI, n_fake), rng.uniform(-spec.eta_max, spec.eta_max, n_fake),
                    fpt, np.where(rng.uniform(size=n_fake) < 0.5, -1.0, 1.0))
    parts = []
    for tk, sel, truth in ((trk, idx, idx), (fk if n_fake else None, np.arange(n_fake), np.full(n_fake, -1))):
        if tk is None or sel.size == 0:
            continue
        k = sel.size
        pts = []
        for rho in PIXEL_R:
            t = tk.cyl_crossings(rho, 1).min(axis=1)
            x, y, z = tk.pos(np.where(np.isfinite(t), t, 0.0))
            x, y, z = x[sel], y[sel], z[sel]
            phi = np.arctan2(y, x) + rng.normal(0.0, SIGMA_PIXEL, k) / rho
            pts.append((rho * np.cos(phi), rho * np.sin(phi), z + rng.normal(0.0, SIGMA_PIXEL, k)))
        rec = {
            "pt": tk.pt[sel] * (1.0 + rng.normal(0.0, 0.02, k)),
            "eta": tk.eta[sel] + rng.normal(0.0, 0.002, k),
            "phi": tk.phi0[sel] + rng.normal(0.0, 0.002, k),
            "vx": tk.xs[sel] + rng.normal(0.0, 0.05, k),
            "vy": tk.ys[sel] + rng.normal(0.0, 0.05, k),
            "vz": tk.z0[sel] + rng.normal(0.0, 0.05, k),
            "x0": pts[0][0], "y0": pts[0][1], "z0": pts[0][2],
            "x1": pts[1][0], "y1": pts[1][1], "z1": pts[1][2],
            "q": tk.q[sel],
            "truth": truth,
        }
        parts.append(rec)
    out = {}
    for f in PLS_FIELDS:
        out[f] = (np.concatenate([p[f] for p in parts]) if parts else np.zeros(0)).astype(np.float32)
    out["q"] = (np.concatenate([p["q"] for p in parts]) if parts else np.zeros(0)).astype(np.int32)
    out["truth"] = (np.concatenate([p["truth"] for p in parts]) if parts else np.zeros(0)).astype(np.int32)
    perm = rng.permutation(out["q"].shape[0])
    return {k: v[perm] for k, v in out.items()}


def generate_event(geom: Geometry, spec: EventSpec, seed: int) -> Event:
    rng = np.random.Generator(np.random.PCG64(seed))
    trk, d0 = _make_tracks(rng, spec)
    x, y, z, sensor, truth = _signal_hits(rng, geom, trk, spec)
    if spec.inefficiency > 0.0:
        keep = rng.uniform(size=x.shape[0]) >= spec.inefficiency
        x, y, z, sensor, truth = x[keep], y[keep], z[keep], sensor[keep], truth[keep]
    if spec.noise is not None:
        n_noise = int(spec.noise[1]) if spec.noise[0] == "count" else int(round(spec.noise[1] * x.shape[0]))
        nx, ny, nz, ns = _noise_hits(rng, geom, n_noise, spec)
        x = np.concatenate([x, nx])
        y = np.concatenate([y, ny])
        z = np.concatenate([z, nz])
        sensor = np.concatenate([sensor, ns])
        truth = np.concatenate([truth, np.full(n_noise, -1, dtype=np.int64)])
    perm = rng.permutation(x.shape[0])
    ev = Event(
        x=x[perm].astype(np.float32), y=y[perm].astype(np.float32), z=z[perm].astype(np.float32),
        sensor=sensor[perm].astype(np.int32), truth=truth[perm].astype(np.int32),
        trk={"pt": trk.pt, "eta": trk.eta, "phi": trk.phi0, "q": trk.q, "z0": trk.z0, "d0": d0},
    )
    if spec.seeds:
        ev.pls = _make_seeds(rng, trk, d0, spec)
    return ev


def concat_events(events):
    """Concatenate events into one batch: SoA arrays plus ``hit_offsets`` / ``pls_offsets`` (int32, n+1)."""
    hit_off = np.concatenate([[0], np.cumsum([e.n_hits for e in events])]).astype(np.int32)
    pls_off = np.concatenate([[0], np.cumsum([e.n_pls for e in events])]).astype(np.int32)
    batch = {
        "x": np.concatenate([e.x for e in events]),
        "y": np.concatenate([e.y for e in events]),
        "z": np.concatenate([e.z for e in events]),
        "sensor": np.concatenate([e.sensor for e in events]),
        "hit_offsets": hit_off,
        "pls_offsets": pls_off,
        "pls": {},
    }
    if pls_off[-1] > 0:
        for f in PLS_FIELDS + ("q",):
            dt = np.int32 if f == "q" else np.float32
            batch["pls"][f] = np.concatenate(
                [e.pls[f] if e.pls else np.zeros(0, dtype=dt) for e in events]
            ).astype(dt)
    return batch
