"""Build the C-ABI shared library in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_06641_b200.build [--force] [--verbose]

Output: paper_2606_06641_b200/libafsat_b200.so (git-ignored; travels to the GPU box with gpurun).
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libafsat_b200.so"
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

SOURCES_CU = [CSRC / "afsat.cu", CSRC / "afsat_ks32.cu"]
SOURCES_CPP = [CSRC / "precompute.cpp", CSRC / "parser.cpp"]
DEPS = [CSRC / "afsat_kernels.cuh", CSRC / "afsat_split.cuh", CSRC / "afsat_step.cuh", CSRC / "afsat_internal.h",
        PKG.parent / "include" / "afsat.h"]

# the two CUDA translation units are compiled in parallel
# -static-global-template-stub=false: a kernel template instantiated in one unit is launched from the other
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-static-global-template-stub=false", "-Xcompiler", "-fPIC"]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES_CU + SOURCES_CPP + DEPS + [Path(__file__)])


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    objdir = PKG / "build"
    objdir.mkdir(exist_ok=True)
    objs = []
    for src in SOURCES_CPP:
        obj = objdir / (src.stem + ".o")
        cmd = ["g++", "-O2", "-std=gnu++17", "-fPIC", "-c", str(src), "-o", str(obj)]
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.check_call(cmd)
        objs.append(obj)
    procs = []
    for src in SOURCES_CU:                                            # the CUDA translation units in parallel
        obj = objdir / (src.stem + ".o")
        cmd = [NVCC, *NVCC_FLAGS, *os.environ.get("AFSAT_NVCC_FLAGS", "").split(), "-c", str(src), "-o", str(obj)]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd), flush=True)
        procs.append((cmd, subprocess.Popen(cmd)))
        objs.append(obj)
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise subprocess.CalledProcessError(pr.returncode, cmd)
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp),
           *map(str, objs), "-lquadmath", "-cudart", "static"]
    if verbose:
        print(" ".join(cmd), flush=True)
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
