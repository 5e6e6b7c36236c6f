"""Build ``libgenga_b200.so`` (the C-ABI CUDA library, include/genga.h) for sm_100a with nvcc.

The library is built IN-TREE next to this file (``paper_2309_08217_b200/libgenga_b200.so``) so
that it travels with the repository snapshot to the GPU box.  nvcc cross-compiles without a GPU.

    python -m paper_2309_08217_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
LIB_PATH = os.path.join(_HERE, "libgenga_b200.so")
_OBJ_DIR = os.path.join(_HERE, "build")

SOURCES = ["api.cu", "prep.cu", "fused_step.cu", "mega_step.cu", "lean_step.cu", "kick_fp32.cu", "kick_fp64.cu", "nearfield.cu", "drift.cu", "reduce.cu", "merge.cu", "probe.cu", "noalloc.cu"]
HEADERS = ["genga_internal.cuh", "tile_pipeline.cuh", "momentum.cuh", "kepler.cuh", "prep_tile.cuh",
           "kick32_body.cuh", "kick64_body.cuh", "kick_sym_body.cuh", "nearfield_body.cuh", "onbody_body.cuh", "encounter.cuh"]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "--fmad=true"]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")
    return exe


def _newest_header() -> float:
    paths = [os.path.join(_CSRC, h) for h in HEADERS] + [os.path.join(_INC, "genga.h"), os.path.abspath(__file__)]
    return max(os.path.getmtime(p) for p in paths)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile every .cu to an object (only the stale ones) and link the shared library.
    ``GENGA_NVCC_EXTRA`` (environment, space separated) appends flags, e.g. ``-DGENGA_SYM_STATS`` for the
    cycle counters of the symmetric kernels (a debugging build; pass --force with it)."""
    nvcc = _nvcc()
    extra = os.environ.get("GENGA_NVCC_EXTRA", "").split()
    os.makedirs(_OBJ_DIR, exist_ok=True)
    hdr_t = _newest_header()
    objs, procs = [], []
    for src in SOURCES:
        s = os.path.join(_CSRC, src)
        o = os.path.join(_OBJ_DIR, src.replace(".cu", ".o"))
        objs.append(o)
        if force or not os.path.exists(o) or os.path.getmtime(o) < max(os.path.getmtime(s), hdr_t):
            cmd = [nvcc, *NVCC_FLAGS, *extra, "-I", _INC, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas")
                cmd.insert(2, "-v")
                print(" ".join(cmd), flush=True)
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = []
    for src, p in procs:
        out, _ = p.communicate()
        if verbose and out:
            print(out, flush=True)
        if p.returncode != 0:
            failed.append((src, out))
    if failed:
        raise RuntimeError("nvcc failed:\n" + "\n".join(f"--- {s} ---\n{o}" for s, o in failed))
    if procs or force or not os.path.exists(LIB_PATH):
        cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", *objs, "-o", LIB_PATH]
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.run(cmd, check=True)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
