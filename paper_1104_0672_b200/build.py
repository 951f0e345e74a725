"""Builds libarkcos.so in-tree with nvcc for sm_100a (python -m paper_1104_0672_b200.build).

One object per translation unit under paper_1104_0672_b200/build/ (git-ignored), recompiled only when the source or a
header it may include is newer; then one link step."""
from __future__ import annotations

import os
import re
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
UNITS = ["arkcos_host.cu", "arkcos_band_tc.cu", "arkcos_fft3.cu", "arkcos_legendre.cpp"]
OBJ_DIR = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libarkcos.so")


def _stale(target: str, deps) -> bool:
    return not os.path.exists(target) or any(os.path.getmtime(target) < os.path.getmtime(d) for d in deps)


def _deps(path: str, seen=None) -> set:
    """The file and every header it includes with quotes, recursively."""
    seen = set() if seen is None else seen
    path = os.path.normpath(path)
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    for m in re.finditer(r'^\s*#include\s+"([^"]+)"', open(path).read(), re.M):
        _deps(os.path.join(os.path.dirname(path), m.group(1)), seen)
    return seen


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    objs = []
    for unit in UNITS:
        src = os.path.join(CSRC, unit)
        obj = os.path.join(OBJ_DIR, os.path.splitext(unit)[0] + ".o")
        objs.append(obj)
        if force or _stale(obj, _deps(src)):
            cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
                   "-Xcompiler", "-fPIC", "-c", "-o", obj, src]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            subprocess.check_call(cmd)
    if force or _stale(LIB, objs):
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
