"""CPU oracle of the LST object-building chain -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The product path
(``paper_2407_18231_b200``) never does.  The arithmetic lives in ``lst_oracle.c``
(plain C, binary32, CUTS.md transcribed); this file is a ctypes loader.
"""
from .binding import (  # noqa: F401
    STAGES,
    KINDS,
    build,
    default_params,
    derived,
    g,
    kappa3,
    md_test,
    ls_test,
    t3_test,
    t5_test,
    t4_test,
    dedup_t4,
    pt_test,
    run_event,
    dedup,
    Params,
)
