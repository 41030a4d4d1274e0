"""The C-ABI boundary without a GPU: the library loads, exports every function include/lst.h
declares, its host-only entry points behave as the header says, and the product path fails loudly
(status codes, no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lst():
    from paper_2407_18231_b200 import build

    build.build()
    import paper_2407_18231_b200 as m

    return m


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "lst.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lst_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lst):
    names = _declared_functions()
    assert "lst_load_geometry" in names and "lst_run_event" in names and "lst_free" in names
    assert sorted(lst.ABI_SYMBOLS) == names, "binding.ABI_SYMBOLS and include/lst.h disagree"
    lib = C.CDLL(lst.library_path())
    for n in names:
        assert hasattr(lib, n), n


def test_no_torch_and_no_oracle_in_the_product_path():
    pkg = os.path.join(ROOT, "paper_2407_18231_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inl", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "lst_oracle" not in text, f
    hdr = open(os.path.join(ROOT, "include", "lst.h")).read()
    assert "torch" not in hdr and "at::" not in hdr


def test_default_params_are_the_cuts_md_table(lst):
    p = lst.lst_default_params().as_dict()
    text = open(os.path.join(ROOT, "CUTS.md")).read()
    rows = dict(re.findall(r"^\| `([A-Z0-9_]+)` \| ([0-9.e+-]+) \|", text, flags=re.M))
    assert len(rows) == 24   # 20 of sections 3-8 + 4 of the extensions (sections 10, 11)
    for name, val in rows.items():
        assert p[name.lower()] == float(np.float32(float(val))), name
    assert p["stage_mask"] == 0x3F


def test_strerror_and_caps(lst):
    lib = C.CDLL(lst.library_path())
    lib.lst_strerror.restype = C.c_char_p
    msgs = {s: lib.lst_strerror(s).decode() for s in (0, -1, -2, -3, -4, 99)}
    assert msgs[0] == "ok" and "capacity" in msgs[-3] and "unknown" in msgs[99]
    assert len(set(msgs.values())) == 6
    caps = lst.lst_default_caps()
    assert caps.max_events == 16 and caps.max_hits >= 16 * 150_000
    b1 = lst.lst_workspace_bytes(caps, 9512)
    b2 = lst.lst_workspace_bytes(lst.lst_default_caps(max_events=32), 9512)
    assert 0 < b1 < b2 < 8 << 30  # a few hundred MB of the B200's 180 GB
    assert lst.lst_workspace_bytes(lst.lst_default_caps(max_md=0), 9512) == 0
    assert lst.lst_workspace_bytes(caps, 0) == 0


def test_argument_errors_are_reported_before_any_cuda_call(lst):
    mods = np.zeros((3, 4), np.int32)
    with pytest.raises(lst.LstError) as e:
        lst.lst_load_geometry(mods, [1, 1, 1, 1], [])  # offsets[0] != 0
    assert e.value.status == lst.LST_ERR_GEOMETRY
    with pytest.raises(lst.LstError) as e:
        lst.lst_load_geometry(mods, [0, 1, 1, 2], [0, 7])  # target out of range
    assert e.value.status == lst.LST_ERR_GEOMETRY
    bad = mods.copy()
    bad[1, 0] = 5  # subdet must be 0 or 1
    with pytest.raises(lst.LstError) as e:
        lst.lst_load_geometry(bad, [0, 0, 0, 0], [])
    assert e.value.status == lst.LST_ERR_GEOMETRY
    with pytest.raises(lst.LstError) as e:
        lst.lst_load_geometry(mods, [0, 2, 1, 1], [0, 1])  # decreasing offsets
    assert e.value.status == lst.LST_ERR_GEOMETRY
    for bad_rel in (1e-4, 1.1e-5, -1e-6, float("nan")):  # the near window the pre-filters are sized for: [0, 1e-5]
        with pytest.raises(lst.LstError) as e:
            lst.lst_load_geometry(mods, [0, 0, 0, 0], [], lst.lst_default_params(near_rel=bad_rel))
        assert e.value.status == lst.LST_ERR_ARG
    lst.lst_free(None)  # NULL is a no-op


def test_scan_entry_points_check_their_arguments_first(lst):
    """n < 0, NULL / misaligned pointers and n beyond the fixed limit are turned down before any CUDA call."""
    from paper_2407_18231_b200 import binding

    lib = binding._lib()
    buf = C.c_void_p(4096)  # never dereferenced
    for f in (lib.lst_scan_counts, lib.lst_scan_counts_static):
        assert f(buf, -1, buf, None) == lst.LST_ERR_ARG
        assert f(buf, 8, None, None) == lst.LST_ERR_ARG
        assert f(None, 8, buf, None) == lst.LST_ERR_ARG
        assert f(C.c_void_p(4100), 8, buf, None) == lst.LST_ERR_ARG  # counts must be 16-byte aligned
    assert lib.lst_scan_counts_static(buf, lst.LST_SCAN_STATIC_MAX_N + 1, buf, None) == lst.LST_ERR_LIMIT
    assert "LST_SCAN_STATIC_MAX_N" in lib.lst_strerror(lst.LST_ERR_LIMIT).decode()
    hdr = open(os.path.join(ROOT, "include", "lst.h")).read()
    assert re.search(r"#define LST_SCAN_STATIC_MAX_N \(1 << 24\)", hdr) and lst.LST_SCAN_STATIC_MAX_N == 1 << 24


def test_no_gpu_means_an_error_not_a_fallback(lst):
    import torch

    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only box")
    mods = np.zeros((3, 4), np.int32)
    with pytest.raises(lst.LstError) as e:
        lst.lst_load_geometry(mods, [0, 1, 1, 1], [1])
    assert e.value.status == lst.LST_ERR_CUDA


def test_missing_library_raises(lst, monkeypatch):
    from paper_2407_18231_b200 import binding

    monkeypatch.setattr(binding, "_LIB", None)
    monkeypatch.setattr(binding, "_SO", os.path.join(ROOT, "does_not_exist.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.lst_default_params()
