"""Build the CUDA C-ABI library (`libsdf_b200.so`) in-tree with nvcc for sm_100a.

    python -m paper_1903_00353_b200.build [--force]

nvcc cross-compiles without a GPU.  The shared object sits next to this file (it is
git-ignored but travels to the GPU box with the repository snapshot).
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libsdf_b200.so")
SOURCES = ["api.cu", "features.cu", "compute.cu", "fill.cu", "stl_io.cu", "peaks.cu"]
RDC_SOURCES = ["cdp.cu"]          # device-side launches (the dynamic-parallelism ablation): relocatable device code
HEADERS = ["common.cuh", "primitives.cuh", "evaluate.cuh", "tile_features.cuh", os.path.join("..", "..", "include", "sdf.h")]
ARCH_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ARCH_FLAGS + ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
LINK_FLAGS = ARCH_FLAGS + ["-shared", "-Xcompiler", "-fPIC", "--cudart", "static", "-lcudadevrt"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def source_hash() -> str:
    """Content hash of everything the library is built from (mtimes do not survive the
    snapshot copy to the GPU box)."""
    import hashlib
    h = hashlib.sha256()
    h.update(" ".join(NVCC_FLAGS + LINK_FLAGS).encode())
    for s in SOURCES + RDC_SOURCES + HEADERS:
        with open(os.path.join(CSRC, s), "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(LIB + ".hash"):
        return True
    with open(LIB + ".hash") as f:
        return f.read().strip() != source_hash()


def build_library(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    # one object per source (compiled side by side), cdp.cu alone as relocatable device code; the
    # final nvcc link runs the device link for it and leaves the other objects as they are
    import tempfile
    extra = ["-Xptxas", "-v"] if verbose else []
    with tempfile.TemporaryDirectory(prefix="sdf_b200_build_") as tmp:
        jobs, objs = [], []
        for s in SOURCES + RDC_SOURCES:
            obj = os.path.join(tmp, os.path.splitext(s)[0] + ".o")
            rdc = ["-rdc=true"] if s in RDC_SOURCES else []
            jobs.append(subprocess.Popen([_nvcc()] + NVCC_FLAGS + rdc + extra + ["-c", os.path.join(CSRC, s), "-o", obj]))
            objs.append(obj)
        rcs = [j.wait() for j in jobs]
        if any(rcs):
            raise subprocess.CalledProcessError(max(rcs), "nvcc -c")
        subprocess.check_call([_nvcc()] + LINK_FLAGS + ["-o", LIB] + objs)
    with open(LIB + ".hash", "w") as f:
        f.write(source_hash())
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
