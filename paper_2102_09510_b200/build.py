"""Builds libxs_b200.so in-tree with nvcc for sm_100a (no JIT cache, the .so travels with the repo)."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(_HERE, "libxs_b200.so")
OBJ = os.path.join(_HERE, "_obj")      # object cache (git-ignored); sources compile in parallel
SOURCES = ["xs_api.cu", "xs_kernels.cu", "xs_sweep_static.cu", "xs_sweep_clause.cu", "xs_sweep_warp.cu", "xs_static.cu", "xs_diag.cu", "xs_graph.cpp", "xs_stats.cpp"] + \
          [f"xs_sweep_static_i{cw}{nc}.cu" for cw in (1, 2) for nc in (1, 2, 4)] + \
          [f"xs_sweep_clause_r{r}.cu" for r in range(4, 17)]
HEADERS = ["xs_internal.h", "xs_device.cuh", "xs_sweep_static.cuh", "xs_sweep_clause.cuh", os.path.join("..", "..", "include", "xs.h")]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libxs_b200.so cannot be built")


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return SO
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
             "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]
    if verbose:
        flags.append("-Xptxas=-v")
    t_hdr = max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)

    def compile_one(src: str) -> str:
        obj = os.path.join(OBJ, src + ".o")
        path = os.path.join(CSRC, src)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(t_hdr, os.path.getmtime(path)):
            subprocess.check_call([nvcc] + flags + ["-c", path, "-o", obj])
        return obj

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as pool:
        objs = list(pool.map(compile_one, SOURCES))
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-o", SO] + objs)
    return SO


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
