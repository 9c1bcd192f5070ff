"""Build the CUDA library libemx.so in-tree for sm_100a (nvcc cross-compiles without a GPU).

    python -m paper_2203_09467_b200.build [--force]

-fmad=false: fp64 multiplies and adds are not contracted into FMAs, so +, -, *, /, sqrt round exactly as
IEEE prescribes in source order (DESIGN.md section 6 explains why parity wants this and what it costs).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SRC = ["emx_api.cu", "emx_kernels.cu", "emx_transport.cu"]
LIB = os.path.join(HERE, "libemx.so")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
         "-Xcompiler", "-fPIC", "-shared", "--cudart", "static"]


def build(force=False, extra=()):
    srcs = [os.path.join(CSRC, s) for s in SRC]
    deps = srcs + [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".h")]
    deps.append(os.path.join(HERE, "..", "include", "emx.h"))
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + FLAGS + list(extra) + ["-o", LIB] + srcs
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
