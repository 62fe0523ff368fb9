"""Build the C-ABI library `libdg_b200.so` (include/dg.h) in-tree with nvcc for sm_100a.

    python -m paper_2208_11131_b200.build [--force]

The stage kernels are compiled once per (dim, m, tracer row or not) in parallel (32 translation units of
dg_stage_inst.cu);
objects land in paper_2208_11131_b200/build/ and are rebuilt only when a source is newer.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libdg_b200.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH + ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC"]


def _nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the DG library cannot be built (there is no CPU fallback)")
    return exe


def _sources_mtime():
    return max(os.path.getmtime(os.path.join(CSRC, f)) for f in os.listdir(CSRC)) if os.path.isdir(CSRC) else 0.0


def _compile(job):
    out, cmd = job
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), r.stderr))
    return out


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile and link the library if it is missing or older than its sources; returns its path."""
    newest = max(_sources_mtime(), os.path.getmtime(os.path.join(HERE, "..", "include", "dg.h")))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    nvcc = _nvcc()
    os.makedirs(OBJ, exist_ok=True)
    jobs = []
    for t in (0, 1):            # without / with the passive-tracer row
        for d in (2, 3):
            for m in range(1, 9):
                o = os.path.join(OBJ, "stage_%d_%d%s.o" % (d, m, "_t1" if t else ""))
                jobs.append((o, [nvcc] + NVCC_FLAGS + ["-DDG_DIM=%d" % d, "-DDG_M=%d" % m, "-DDG_TRACER=%d" % t, "-c",
                                                      os.path.join(CSRC, "dg_stage_inst.cu"), "-o", o]))
    o = os.path.join(OBJ, "api.o")
    jobs.append((o, [nvcc] + NVCC_FLAGS + ["-c", os.path.join(CSRC, "dg_api.cu"), "-o", o]))
    o = os.path.join(OBJ, "tables.o")
    jobs.append((o, [nvcc] + NVCC_FLAGS + ["-x", "cu", "-c", os.path.join(CSRC, "dg_tables.cpp"), "-o", o]))
    todo = [j for j in jobs if force or not os.path.exists(j[0]) or os.path.getmtime(j[0]) < newest]
    # heaviest (3D, large m) first
    todo.sort(key=lambda j: j[0], reverse=True)
    with ThreadPoolExecutor(max_workers=max(1, (os.cpu_count() or 4))) as ex:
        for out in ex.map(_compile, todo):
            if verbose:
                print("built", os.path.relpath(out, HERE))
    cmd = [nvcc] + ARCH + ["-shared", "-o", LIB] + [j[0] for j in jobs]
    _compile((LIB, cmd))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
