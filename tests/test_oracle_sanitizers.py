"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (CPU only).

compute-sanitizer is closed on the GPU pool, so the host side is the sanitizer coverage there is: the
oracle's C source is built with -fsanitize=address,undefined -fno-sanitize-recover=all and driven through
its pins, the duplicate-removal cases and whole events (C1, C2, C4, empty, rejected input) in a subprocess
with libasan preloaded.  A second build with a deliberate one-element under-allocation must be caught,
which shows the instrumentation is live.
"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "lst_oracle.c")
RUNNER = os.path.join(ROOT, "tests", "oracle_sanitized_run.py")


def _libasan():
    p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    return p if os.path.isabs(p) and os.path.exists(p) else None


def _build(tmp_path, src_text, name):
    c = tmp_path / (name + ".c")
    c.write_text(src_text)
    (tmp_path / "lst_oracle.h").write_text(open(os.path.join(ROOT, "oracle", "lst_oracle.h")).read())
    so = str(tmp_path / (name + ".so"))
    subprocess.run(["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                    "-fno-omit-frame-pointer", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-shared", "-fPIC",
                    "-o", so, str(c), "-lm"], check=True)
    return so


def _run(so):
    env = dict(os.environ, LD_PRELOAD=_libasan(), ASAN_OPTIONS="detect_leaks=0:abort_on_error=0",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    return subprocess.run([sys.executable, RUNNER, so], capture_output=True, text=True, env=env, timeout=600)


@pytest.mark.skipif(_libasan() is None, reason="gcc's libasan.so not found")
def test_oracle_clean_under_asan_ubsan(tmp_path):
    r = _run(_build(tmp_path, open(SRC).read(), "lst_oracle"))
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, r.stdout[-2000:] + r.stderr[-4000:]
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr


@pytest.mark.skipif(_libasan() is None, reason="gcc's libasan.so not found")
def test_sanitizer_is_live(tmp_path):
    src = open(SRC).read()
    old = "int* s_first = (int*)calloc((size_t)(2 * n_modules + 1), sizeof(int));"
    assert src.count(old) == 1
    r = _run(_build(tmp_path, src.replace(old, "int* s_first = (int*)calloc((size_t)(2 * n_modules), sizeof(int));"),
                    "lst_oracle"))
    assert r.returncode != 0 and ("AddressSanitizer" in r.stderr or "runtime error" in r.stderr)
