"""Build libpff.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2606_23458_b200.build [--force] [--trace]

nvcc cross-compiles without a GPU.  The built library stays next to this file (git-ignored, but it
travels with the repo snapshot to the GPU box).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libpff.so")
LIB_TRACE = os.path.join(HERE, "libpff_trace.so")
SOURCES = ["mesh_setup.cpp", "pff_api.cu", "pff_step.cu", "pff_damage.cu", "pff_energy.cu", "pff_host.cu", "pff_equilibrium.cu", "pff_multigrid.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def _deps_mtime() -> float:
    files = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(ROOT, "include", "pff.h")]
    return max(os.path.getmtime(f) for f in files)


def _compile(src: str, verbose: bool, trace: bool = False) -> str:
    obj = os.path.join(OBJ, os.path.splitext(src)[0] + (".trace.o" if trace else ".o"))
    cmd = [NVCC, *FLAGS, *(["-DPFF_TRACE"] if trace else []), "-c", os.path.join(CSRC, src), "-o", obj]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{r.stdout}\n{r.stderr}")
    if verbose:
        print(r.stderr)
    return obj


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    """trace=True builds libpff_trace.so: the same sources with -DPFF_TRACE (phase timestamps, pff_trace_set)."""
    lib = LIB_TRACE if trace else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= _deps_mtime():
        return lib
    os.makedirs(OBJ, exist_ok=True)
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(lambda s: _compile(s, verbose, trace), SOURCES))
    r = subprocess.run([NVCC, "-shared", "-o", lib, *objs, "-gencode", "arch=compute_100a,code=sm_100a"],
                       capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
