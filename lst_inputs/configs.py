"""The five BASELINE.json workloads made concrete.

C1 toy barrel, 20 helices            -> MD..T5 only
C2 barrel, 500 helices + noise + 5%  -> full chain + duplicate removal
C3 PU200-like single event (barrel + endcap, ~7000 helices)
C4 C2 + pLS seeds + 50 displaced helices
C5 batches of 16 C3-like events at PU 50/100/140/200/250 (35 tracks per PU unit)
C6 (not a BASELINE.json config) C5's generator with strip-like sensors: 5 cm strips along z on
   the three outer barrel layers and two strip rows per endcap ring beyond r = 60 cm, with the z windows of the
   cuts opened to the strip length (C6_PARAMS) -- the combinatorics-heavier second workload
C7 C4's event with 15 % hit inefficiency on a connection map with skip-layer edges: run with stage
   mask C7_MASK (T4 objects on) it exercises "more objects" for tracks with a missing layer
"""
from __future__ import annotations

from functools import lru_cache

from .connmap import build_connection_map
from .events import Event, EventSpec, generate_event
from .geometry import Geometry, make_geometry

CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
# cut constants of the strip-like workload: the r-z windows must hold a strip (pitch 5 cm, i.e. +-2.5 cm of
# quantisation per hit); everything else as in CUTS.md section 1
C7_MASK = 0x7f  # every stage of CUTS.md sections 3-8 plus the T4 extension of section 10
STRIP_PITCH = 5.0
C6_PARAMS = {"md_z_tol": 5.5, "ls_z_tol": 4.0, "t3_z_tol0": 4.0, "t3_z_tol1": 1.0, "pt_z_tol": 5.0}
PU_POINTS = (50, 100, 140, 200, 250)
TRACKS_PER_PU = 35

_GEOM_OF = {"C1": "barrel_z60", "C2": "barrel_z60", "C3": "barrel_z120_endcap",
            "C4": "barrel_z60", "C5": "barrel_z120_endcap", "C6": "barrel_z120_endcap", "C7": "barrel_z60"}


@lru_cache(maxsize=None)
def _geometry(name: str, skip: bool = False):
    g = make_geometry(name)
    off, tgt = build_connection_map(g, skip=skip)
    return g, off, tgt


def make_config_geometry(config: str):
    """(Geometry, conn_offsets, conn_targets) of a config."""
    return _geometry(_GEOM_OF[config], config == "C7")


def spec_of(config: str, pu: int = 200, seeds: bool | None = None) -> EventSpec:
    if config == "C1":
        return EventSpec(n_tracks=20, pt_dist=("loguniform", 0.8, 10.0), eta_max=0.8)
    if config == "C2":
        return EventSpec(n_tracks=500, pt_dist=("loguniform", 0.8, 20.0), eta_max=1.0,
                         noise=("count", 2000), inefficiency=0.05)
    if config == "C3" or config == "C5":
        return EventSpec(n_tracks=TRACKS_PER_PU * pu, pt_dist=("power3", 0.3), eta_max=2.5,
                         noise=("frac", 0.01), seeds=bool(seeds))
    if config == "C6":
        return EventSpec(n_tracks=TRACKS_PER_PU * pu, pt_dist=("power3", 0.3), eta_max=2.5,
                         noise=("frac", 0.01), seeds=bool(seeds), strip_pitch=STRIP_PITCH)
    if config == "C4":
        return EventSpec(n_tracks=500, pt_dist=("loguniform", 0.8, 20.0), eta_max=1.0,
                         noise=("count", 2000), inefficiency=0.05, seeds=True, n_displaced=50)
    if config == "C7":
        return EventSpec(n_tracks=500, pt_dist=("loguniform", 0.8, 20.0), eta_max=1.0,
                         noise=("count", 2000), inefficiency=0.15, seeds=True, n_displaced=50)
    raise ValueError(config)


def make_config_event(config: str, pu: int = 200, index: int = 0, seeds: bool | None = None) -> Event:
    """Seed = config number (C1..C4); C5: 1000*PU + event index (G7)."""
    geom, _, _ = make_config_geometry(config)
    if config in ("C5", "C6"):
        seed = 1000 * pu + index
    else:
        seed = int(config[1])
        pu = 200
    return generate_event(geom, spec_of(config, pu, seeds), seed)


def c5_batch(pu: int = 200, n_events: int = 16, seeds: bool = True, first: int = 0, config: str = "C5"):
    return [make_config_event(config, pu=pu, index=first + i, seeds=seeds) for i in range(n_events)]
