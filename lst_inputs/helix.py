"""Helix propagation in a uniform field along z (float64; used only to MAKE inputs).

Conventions: B = 3.8 T along +z, lengths in cm,
momenta in GeV.  Radius R = pT * KR with KR = 100 / (0.3 * B) cm/GeV.  A
particle of charge q turns with sense h = -q (q = +1 turns clockwise seen
from +z, i.e. has NEGATIVE signed curvature in the counter-clockwise-positive
convention).  With turning angle t >= 0 (transverse arc length s = R*t):

    dir(t) = phi0 + h*t
    x(t) = cx + h*R*sin(dir(t)),  y(t) = cy - h*R*cos(dir(t)),  z(t) = z0 + R*t*sinh(eta)
    (cx, cy) = (xs - h*R*sin(phi0), ys + h*R*cos(phi0))
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

B_FIELD = 3.8
KR = 100.0 / (0.3 * B_FIELD)  # cm per GeV
TWO_PI = 2.0 * np.pi


@dataclass
class Tracks:
    xs: np.ndarray
    ys: np.ndarray
    z0: np.ndarray
    phi0: np.ndarray
    eta: np.ndarray
    pt: np.ndarray
    q: np.ndarray  # +-1

    def __post_init__(self):
        for k in ("xs", "ys", "z0", "phi0", "eta", "pt", "q"):
            setattr(self, k, np.asarray(getattr(self, k), dtype=np.float64))
        self.R = self.pt * KR
        self.h = -self.q
        self.cx = self.xs - self.h * self.R * np.sin(self.phi0)
        self.cy = self.ys + self.h * self.R * np.cos(self.phi0)
        self.sinh_eta = np.sinh(self.eta)

    def __len__(self):
        return self.pt.shape[0]

    def pos(self, t):
        """Position at turning angle ``t`` (broadcast against the track axis 0)."""
        t = np.asarray(t, dtype=np.float64)
        ex = (slice(None),) + (None,) * (t.ndim - 1)
        d = self.phi0[ex] + self.h[ex] * t
        x = self.cx[ex] + self.h[ex] * self.R[ex] * np.sin(d)
        y = self.cy[ex] - self.h[ex] * self.R[ex] * np.cos(d)
        z = self.z0[ex] + self.R[ex] * t * self.sinh_eta[ex]
        return x, y, z

    def cyl_crossings(self, rho: float, n_turns: int):
        """Turning angles at which the transverse radius equals ``rho``.

        Returns [n_tracks, 2*n_turns], NaN where the circle does not reach rho.
        """
        C = np.hypot(self.cx, self.cy)
        psi = np.arctan2(self.cy, self.cx)
        with np.errstate(divide="ignore", invalid="ignore"):
            w = (rho * rho - C * C - self.R * self.R) / (2.0 * self.h * self.R * C)
        ok = np.abs(w) <= 1.0
        a = np.arcsin(np.where(ok, w, 0.0))
        d1 = psi + a
        d2 = psi + np.pi - a
        t1 = np.mod(self.h * (d1 - self.phi0), TWO_PI)
        t2 = np.mod(self.h * (d2 - self.phi0), TWO_PI)
        out = []
        for k in range(n_turns):
            out.append(np.where(ok, t1 + k * TWO_PI, np.nan))
            out.append(np.where(ok, t2 + k * TWO_PI, np.nan))
        return np.stack(out, axis=1)

    def plane_crossing(self, zd: float):
        """Turning angle at which z == zd (NaN if never, i.e. moving away or eta == 0)."""
        with np.errstate(divide="ignore", invalid="ignore"):
            t = (zd - self.z0) / (self.R * self.sinh_eta)
        return np.where(np.isfinite(t) & (t > 0.0), t, np.nan)

    def t_exit(self, r_exit: float, z_exit: float, t_max: float):
        """First turning angle at which the particle leaves r < r_exit, |z| < z_exit."""
        tr = self.cyl_crossings(r_exit, 1)
        tr = np.where(np.isnan(tr), np.inf, tr).min(axis=1)
        with np.errstate(divide="ignore", invalid="ignore"):
            tz = (np.sign(self.sinh_eta) * z_exit - self.z0) / (self.R * self.sinh_eta)
        tz = np.where(np.isfinite(tz) & (tz > 0.0), tz, np.inf)
        return np.minimum(np.minimum(tr, tz), t_max)
