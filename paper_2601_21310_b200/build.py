"""Build libdetham.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
SO = os.path.join(PKG, "libdetham.so")
SOURCES = ["api.cu", "lists.cu", "ham_build.cu", "energy.cu", "ediag.cu", "pt2.cu", "expand.cu"]
HEADERS = ["common.cuh", "enumerate.cuh"]


def _stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(ROOT, "include", "detham.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--extended-lambda",
               "-shared", "-Xcompiler", "-fPIC", "-I" + os.path.join(ROOT, "include")]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        cmd += [os.path.join(CSRC, f) for f in SOURCES] + ["-o", SO]
        subprocess.check_call(cmd)
    return SO


def build_probes(force: bool = False) -> list:
    """Compile the stand-alone microbenchmarks under probes/ (random-slot traffic, appends, store variants) for sm_100a."""
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    src_dir = os.path.join(PKG, "probes")
    out_dir = os.path.join(src_dir, "bin")
    os.makedirs(out_dir, exist_ok=True)
    built = []
    for f in sorted(os.listdir(src_dir)):
        if not f.endswith(".cu"):
            continue
        src, exe = os.path.join(src_dir, f), os.path.join(out_dir, f[:-3])
        if force or not os.path.exists(exe) or os.path.getmtime(src) > os.path.getmtime(exe):
            subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", src, "-o", exe])
        built.append(exe)
    return built


if __name__ == "__main__":
    print(build(force=True, verbose=True))
