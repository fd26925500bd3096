"""Builds libpwa_b200.so (the C-ABI library of include/pwa.h) in-tree with nvcc for sm_100a.

    python -m paper_2403_09225_b200.build [--force] [-v]

nvcc cross-compiles without a GPU.  The translation units are compiled in parallel (the lanes sweep kernel is
instantiated once per helicity count) and linked into one shared library.  Objects and the .so are git-ignored;
the .so travels to the GPU box with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(PKG, "csrc")
OBJ = os.path.join(PKG, "build")
LIB = os.path.join(PKG, "libpwa_b200.so")
# (source, object name, extra defines)
UNITS = [("pwa_api.cu", "pwa_api.o", []), ("pwa_fit.cu", "pwa_fit.o", []), ("pwa_fractions.cu", "pwa_fractions.o", []), ("pwa_sweep_lanes.cu", "pwa_sweep_lanes.o", []), ("pwa_batch.cu", "pwa_batch.o", []), ("pwa_static.cu", "pwa_static.o", [])] + \
        [("pwa_sweep_lanes_inst.cu", f"pwa_sweep_lanes_h{h}.o", [f"-DPWA_LANES_H={h}"]) for h in (1, 2, 3, 4)]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
CFLAGS = [*ARCH, "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC,-O2"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(PKG, "..", "include", "pwa.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = _nvcc()
    extra = os.environ.get("PWA_NVCC_EXTRA", "").split()
    cmds = [[nvcc, *CFLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), *defs, "-c", os.path.join(CSRC, src),
             "-o", os.path.join(OBJ, obj)] for src, obj, defs in UNITS]
    with ThreadPoolExecutor(max_workers=min(len(cmds), os.cpu_count() or 4)) as ex:
        logs = list(ex.map(_run, cmds))
    _run([nvcc, *ARCH, "-shared", "-cudart", "static", *[os.path.join(OBJ, obj) for _, obj, _ in UNITS], "-o", LIB])
    if verbose:
        print("\n".join(logs))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
