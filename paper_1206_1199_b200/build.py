"""Build libotoo.so in-tree for sm_100a (nvcc cross-compiles without a GPU).

    python -m paper_1206_1199_b200.build
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["api.cu", "build.cu", "sort.cu", "gravity.cu", "sph.cu", "probe.cu"]
HEADERS = ["common.cuh", "walk.cuh", "walk_ws.cuh", "grav_eval.cuh", "keys.cuh", os.path.join("..", "..", "include", "otoo.h")]
LIB = os.path.join(HERE, "libotoo.so")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(HERE, "csrc", f) for f in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    flags = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
    flags += os.environ.get("OTOO_NVCC_FLAGS", "").split()      # e.g. -DOTOO_EVAL_UNR=8 for an A/B library
    if verbose:
        flags += ["-Xptxas", "-v"]

    hdr_time = max(os.path.getmtime(os.path.join(HERE, "csrc", h)) for h in HEADERS)

    def compile_one(f: str) -> str:          # one nvcc per translation unit, side by side (no device code crosses files)
        obj = os.path.join(objdir, f.replace(".cu", ".o"))
        src_time = max(hdr_time, os.path.getmtime(os.path.join(HERE, "csrc", f)))
        if not verbose and os.path.exists(obj) and os.path.getmtime(obj) > src_time:
            return obj                       # (an object newer than its source and every header is kept)
        subprocess.run(["nvcc"] + flags + ["-c", os.path.join(HERE, "csrc", f), "-o", obj], check=True)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC", "-shared", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
