"""Compile the CUDA library for sm_100a into paper_2406_15236_b200/libmpc_b200.so (in-tree).

nvcc cross-compiles without a GPU. --fmad=false: no implicit contraction, every fused
multiply-add in the kernels is an explicit fmaf (reading U1)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "csrc", f) for f in ("abi.cu", "sweep.cu", "cell.cu", "reorder.cu", "generic.cu", "observe.cu", "noalloc.cu")]
DEPS = SRC + [os.path.join(HERE, "csrc", "philox.cuh"), os.path.join(HERE, "csrc", "internal.cuh"), os.path.join(HERE, "csrc", "cell.cuh"),
              os.path.join(HERE, "..", "include", "mpc_b200.h")]
LIB = os.path.join(HERE, "libmpc_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "--fmad=false",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "--threads", "0"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SRC
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
