"""Build libipanll.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1706_01420_b200.build [--force]

nvcc cross-compiles without a GPU.  The built library sits next to this file (git-ignored; it
travels to the GPU box with the gpurun snapshot).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libipanll.so")
SOURCES = [os.path.join(CSRC, "ipa_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, n) for n in ("ipa_kernels.cuh", "ipa_prologue.cuh", "ipa_math.cuh", "ipa_fastmath.cuh",
                                                      "ipa_fastmath_tables.inc")] + [
    os.path.join(ROOT, "include", "ipanll.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared",
]


def nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def up_to_date():
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(d) <= t for d in DEPS)


def build(force=False, verbose=False):
    if not force and up_to_date():
        return LIB
    cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-I", os.path.join(ROOT, "include"),
                                                                          "-o", LIB] + SOURCES
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
