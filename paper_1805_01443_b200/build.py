"""Build libdg.so (the C-ABI library of include/dg.h) in-tree with nvcc for sm_100a.

    python -m paper_1805_01443_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdg.so")
SOURCES = ["dg_api.cu", "dg_static.cu"] + [f"dg_stage_m{m}{f}.cu" for m in (5, 4, 3, 2, 1) for f in ("", "f")]
DEPS = SOURCES + ["dg_kernels.cuh", "dg_stage_fh.cuh", "dg_stage_m1fv.cuh", "dg_stage_launch.cuh", "dg_tables.h", "dg_limit.cuh",
                  os.path.join("..", "..", "include", "dg.h")]
OBJ_DIR = os.path.join(HERE, "build")
NVCC_COMPILE = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--extended-lambda", "-Xcompiler", "-fPIC", "-c",
]
# Order 1 (dg_stage_m1fv.cuh) repeats its row body six times so that its row buffers rotate by renaming; left to itself
# the compiler contracts a * b + c into an FMA in some copies and not in others, and the result of a row would depend
# on its position in the segment (strips of a decomposed domain would no longer reproduce the undivided domain bitwise).
# Without contraction only the FMAs the source spells out are FMAs, in every copy.
PER_SOURCE = {"dg_stage_m1.cu": ["-fmad=false"], "dg_stage_m1f.cu": ["-fmad=false"]}
NVCC_LINK = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    """Compile every translation unit (in parallel) and link libdg.so."""
    if not (force or needs_build()):
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ_DIR, exist_ok=True)
    procs = []
    for src in SOURCES:
        obj = os.path.join(OBJ_DIR, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_COMPILE, *PER_SOURCE.get(src, []), *extra_flags, *(["-Xptxas", "-v"] if verbose else []),
               os.path.join(CSRC, src), "-o", obj]
        procs.append((src, obj, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    objs = []
    for src, obj, pr in procs:
        out, _ = pr.communicate()
        if verbose or pr.returncode != 0:
            sys.stderr.write(out)
        if pr.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(obj)
    subprocess.check_call([nvcc, *NVCC_LINK, *objs, "-o", LIB])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
