"""Builds libcs.so (the CUDA library behind include/cs.h) in-tree with nvcc for sm_100a.

`python -m paper_2604_08463_b200.build` or `build()`; cross-compiles without a GPU.
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libcs.so")
SOURCES = ["cs_lib.cu"]
HEADERS = ["cs_kmeans.cuh", "cs_cells.cuh", "cs_pipe.cuh", "cs_tables.cuh", "cs_like_sc.cuh", "cs_like_direct.cuh", "cs_math.cuh", "cs_optim.cuh", "cs_internal.h", os.path.join("..", "..", "include", "cs.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--shared",
              "-Xcompiler", "-fPIC,-O2,-fvisibility=hidden", "-Xptxas", "-v", "--use_fast_math=false"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    flags = [f for f in NVCC_FLAGS if f != "--use_fast_math=false"] + os.environ.get("CS_NVCC_EXTRA", "").split()
    out = os.environ.get("CS_LIB_OUT", LIB)
    cmd = [_nvcc()] + flags + ["-o", out] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(_HERE, "build.log"), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + log[-4000:])
    if verbose:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
