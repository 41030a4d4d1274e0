"""Seeded synthetic inputs for the LST hot path (geometry, connection map, events).

This package serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2407_18231_b200/``).  It holds none of the method's arithmetic: no
selection cut, no object building.  It only makes inputs -- module tables,
the module connection map ("precomputed connection maps"), outer
tracker hits and inner-tracker seeds / pLSs --
for the five workloads of BASELINE.json.  The recipe is stated in DESIGN.md
("Input recipe").  The paper's own workload (CMS ttbar + 200 PU on the Phase-2
geometry) is not available; these events stand in for it.
"""
from .geometry import Geometry, make_geometry
from .connmap import build_connection_map
from .events import Event, generate_event, concat_events
from .configs import (
    CONFIG_NAMES,
    make_config_event,
    make_config_geometry,
    c5_batch,
    PU_POINTS,
)

__all__ = [
    "Geometry",
    "make_geometry",
    "build_connection_map",
    "Event",
    "generate_event",
    "concat_events",
    "CONFIG_NAMES",
    "make_config_event",
    "make_config_geometry",
    "c5_batch",
    "PU_POINTS",
]
