"""Build the CUDA library in-tree: paper_2607_00579_b200/libepo.so (sm_100a only).

nvcc cross-compiles without a GPU, so this runs on the CPU-only build box; the resulting .so travels to
the B200 box with the repository snapshot.  Each .cu is compiled to an object under build/ (cached by
modification time) and the objects are linked with the static CUDA runtime.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libepo.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

CFLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
          "-Xcompiler", "-fPIC,-O2,-fvisibility=hidden", "-I", os.path.join(ROOT, "include"), "-I", CSRC]
LFLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-ldl"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + [os.path.join(ROOT, "include", "epo.h"), __file__]


def build(force: bool = False, verbose: bool = False, defines=(), lib_path: str = LIB, obj_tag: str = "") -> str:
    """Compile stale objects and link.  `defines` / `lib_path` / `obj_tag` build a tuning variant elsewhere."""
    os.makedirs(OBJ, exist_ok=True)
    hdr_t = max(os.path.getmtime(h) for h in _headers())
    objs, relink = [], force or not os.path.exists(lib_path)
    for src in sources():
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + obj_tag + ".o")
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), hdr_t):
            cmd = [NVCC] + CFLAGS + [f"-D{d}" for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src]
            subprocess.check_call(cmd)
            relink = True
        objs.append(obj)
    if relink or any(os.path.getmtime(o) > os.path.getmtime(lib_path) for o in objs):
        tmp = lib_path + ".%d.tmp" % os.getpid()
        subprocess.check_call([NVCC] + LFLAGS + ["-o", tmp] + objs)
        os.replace(tmp, lib_path)
    return lib_path


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
