"""Builds the CUDA library (sm_100a only) in-tree: paper_2407_18231_b200/liblst_b200.so.

Flags that matter for parity (CUTS.md section 0): -fmad=false (no FMA contraction), precise
division and square root, no flush-to-zero, no fast-math; host code with -ffp-contract=off.
"""
from __future__ import annotations

import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(_HERE, "liblst_b200.so")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math,-Wall",
    "-shared", "-cudart", "static",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*")) + [os.path.join(INCLUDE, "lst.h"), os.path.abspath(__file__)])


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(SO) and os.path.getmtime(SO) >= max(os.path.getmtime(s) for s in sources()):
        return SO
    return _compile(SO, [], verbose)


def _compile(out: str, defines, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = out + f".tmp{os.getpid()}"
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [f"-D{d}" for d in defines] + \
          ["-I", INCLUDE, "-o", tmp, os.path.join(CSRC, "lst_api.cu")]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


def build_variant(out: str, defines) -> str:
    """A debugging build next to the product (never loaded by the package): the same sources with extra -D macros,
    e.g. LST_DEBUG_SYNC (waits and prints before every kernel) or the reproducer of profiles/r03_rule3_fault.md."""
    return _compile(os.path.abspath(out), list(defines))


if __name__ == "__main__":
    import sys
    if "--variant" in sys.argv:  # python -m paper_2407_18231_b200.build --variant OUT.so MACRO [MACRO ...]
        i = sys.argv.index("--variant")
        print(build_variant(sys.argv[i + 1], sys.argv[i + 2:]))
    else:
        print(build(force=True, verbose="-v" in sys.argv))
