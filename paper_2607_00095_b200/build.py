"""Build libsnap.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

The translation units are compiled in parallel (`nvcc -c`, one process each) and linked into
`paper_2607_00095_b200/libsnap.so`; object files live in `paper_2607_00095_b200/build/` (git-ignored)."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsnap.so")
SOURCES = ["api.cu", "proj1d_burgers.cu", "proj1d_burgers_fused.cu", "proj1d_fisher.cu", "proj1d_fisher_fused.cu", "proj1d_fluxk.cu", "proj2d.cu", "proj2d_direct.cu", "proj1d_f32.cu"]
HEADERS = ["snap_internal.h", "launch.h", "device_utils.cuh", "kernels_1d.cuh", "kernels_1d_fused.cuh", "kernels_1d_fluxk.cuh", "tridiag.cuh", "kernels_2d.cuh", "kernels_2d_direct.cuh", "kernels_misc.cuh", "kernels_ns.cuh", "kernels_1d_f32.cuh",
           os.path.join("..", "..", "include", "snap.h")]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    flags = ARCH + ["-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC"]
    if verbose:
        flags += ["-Xptxas", "-v"]

    def compile_one(src: str) -> str:
        obj = os.path.join(OBJ, os.path.splitext(src)[0] + ".o")
        subprocess.run([nvcc] + flags + ["-c", os.path.join(CSRC, src), "-o", obj], check=True)
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.run([nvcc] + ARCH + ["-shared", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
