"""In-tree build of libwhp.so (the C-ABI library of include/whp.h) for sm_100a.

    python -m paper_2110_13693_b200.build [--force]

nvcc cross-compiles without a GPU. The .so stays in this directory (git-ignored; it travels
to the GPU box with the tree).
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libwhp.so")
SOURCES = ["whp_api.cu", "whp_eval.cu", "whp_fast.cu", "whp_swaps.cu", "whp_argmin.cu", "whp_nhatc.cu", "whp_legsum.cu", "whp_kmeans.cu", "whp_route.cu", "whp_static.cu"]
HEADERS = ["whp_internal.cuh", "whp_walk.cuh", os.path.join("..", "..", "include", "whp.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=false",  # D6: every fp64 product and sum individually rounded
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libwhp.so cannot be built")


def stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", SO,
               *[os.path.join(CSRC, f) for f in SOURCES]]
        subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
