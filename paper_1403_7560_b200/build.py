"""Build libsw_b200.so (hand-written CUDA for sm_100a + the C ABI of include/sw.h) in-tree.

Usage: python -m paper_1403_7560_b200.build [--force]      (also called by __graft_entry__.build())
nvcc cross-compiles without a GPU; the built .so travels to the GPU box with the repo snapshot.
"""
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsw_b200.so")
SOURCES = [os.path.join(CSRC, "sw_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "sw_kernels.cuh"), os.path.join(CSRC, "sw_rows.cuh"), os.path.join(CSRC, "sw_small.cuh"), os.path.join(ROOT, "include", "sw.h")]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", shutil.which("nvcc")):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libsw_b200 cannot be built (there is no CPU fallback)")


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [nvcc_path(), "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-o", LIB] + SOURCES
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    cmd[1:1] = os.environ.get("SW_B200_NVCC_FLAGS", "").split()   # developer knob: extra -D... for experiments
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
