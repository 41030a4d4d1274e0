"""Runs the oracle's pins and whole events on a library built with -fsanitize=address,undefined.

Started by tests/test_oracle_sanitizers.py as a subprocess with libasan preloaded (the interpreter is not
instrumented, the oracle's C code is).  argv[1] = path of the instrumented shared library.
"""
import importlib.util
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    so = sys.argv[1]
    spec = importlib.util.spec_from_file_location("oracle_sanitized", os.path.join(ROOT, "oracle", "binding.py"))
    O = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(O)
    O.build = lambda force=False: so

    import numpy as np

    from lst_inputs import make_config_event, make_config_geometry
    from tests import test_oracle_dedup as D
    from tests import test_oracle_values as V

    for check in V.CHECKS:
        check(O)
    for name in dir(D):
        if name.startswith("test_") and name != "test_survivors_do_not_overlap_on_c4":
            getattr(D, name)(O)
    n_tc = 0
    for cfg, mask in (("C1", 0x0f), ("C2", 0x2f), ("C4", 0x3f)):
        geom, off, tgt = make_config_geometry(cfg)
        ev = make_config_event(cfg)
        r = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, O.default_params(stage_mask=mask))
        n_tc += len(r["tc"])
    geom, off, tgt = make_config_geometry("C1")
    e = np.zeros(0, np.float32)
    O.run_event(geom.subdet, off, tgt, e, e, e, np.zeros(0, np.int32))            # empty event
    try:
        O.run_event(geom.subdet, off, tgt, [1.0], [2.0], [3.0], [2 * geom.n_modules])  # rejected input
    except ValueError:
        pass
    print("sanitized oracle ok", n_tc)


if __name__ == "__main__":
    main()
