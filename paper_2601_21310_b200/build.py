"""Build libdetham.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
SO = os.path.join(PKG, "libdetham.so")
SO_CHECKED = os.path.join(PKG, "libdetham_checked.so")  # -DDETHAM_CHECKED: device asserts at every computed index (common.cuh)
SOURCES = ["api.cu", "lists.cu", "ham_build.cu", "pair_build.cu", "energy.cu", "energy_static.cu", "ediag.cu", "pt2.cu", "pt2_stream.cu", "expand.cu"]
HEADERS = ["common.cuh", "enumerate.cuh", "pt2_common.cuh"]


def _stale(so: str = SO) -> bool:
    if not os.path.exists(so):
        return True
    t = os.path.getmtime(so)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "detham.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    so = SO_CHECKED if checked else SO
    if force or _stale(so):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--extended-lambda",
               "-shared", "-Xcompiler", "-fPIC", "-I" + os.path.join(ROOT, "include")]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        if checked:
            cmd += ["-DDETHAM_CHECKED"]
        cmd += [os.path.join(CSRC, f) for f in SOURCES] + ["-o", so]
        subprocess.check_call(cmd)
    return so


if __name__ == "__main__":
    print(build(force=True, verbose=True))
