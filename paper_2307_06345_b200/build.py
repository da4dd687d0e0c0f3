"""Build libcornerstone_b200.so (hand-written CUDA for sm_100a) in-tree with nvcc.

    python -m paper_2307_06345_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so lands next to this file so that it travels
with the repository snapshot to the GPU box; object files go to csrc/build/.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libcornerstone_b200.so")
SOURCES = ["cs_context.cu", "cs_particles.cu", "cs_sort.cu", "cs_leaves.cu", "cs_leaves_direct.cu", "cs_link.cu", "cs_props.cu", "cs_global.cu", "cs_static.cu", "cs_api.cu", "cs_api32.cu"]
HEADERS = ["cs_internal.cuh", "cs_device.cuh", os.path.join("..", "..", "include", "cornerstone.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-Xptxas", "-warn-spills"]
# tuning overrides for experiments, e.g. CS_DEFINES="-DCS_SORT_BLOCK=384 -DCS_SORT_ITEMS=20"
FLAGS += os.environ.get("CS_DEFINES", "").split()


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _compile(src: str, force: bool, verbose: bool) -> str:
    s = os.path.join(CSRC, src)
    o = os.path.join(OBJ, src.replace(".cu", ".o"))
    if (not force and os.path.exists(o)
            and os.path.getmtime(o) >= max(os.path.getmtime(s), _newest_header())):
        return o
    cmd = [NVCC] + FLAGS + ["-c", s, "-o", o]
    r = subprocess.run(cmd, capture_output=True, text=True)
    with open(o + ".log", "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}")
    return o


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(lambda s: _compile(s, force, verbose), SOURCES))
    if (force or not os.path.exists(LIB)
            or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs)):
        cmd = [NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + objs + ["-cudart", "static"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
