"""Builds libidfx.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2304_13746_b200.build [--force]
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = [os.path.join(_HERE, "csrc", "idfx.cu"), os.path.join(_HERE, "csrc", "probe.cu")]
HEADERS = sorted(os.path.join(_HERE, "csrc", f) for f in os.listdir(os.path.join(_HERE, "csrc")) if f.endswith(".cuh")) + [
    os.path.join(os.path.dirname(_HERE), "include", "idfx.h"), os.path.join(os.path.dirname(_HERE), "include", "idfx_probe.h")]
LIB = os.path.join(_HERE, "libidfx.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
    "-split-compile", "0",   # the kernels of one translation unit are optimised in parallel (same code, half the build time)
]


def build(force=False, verbose=False):
    deps = SOURCES + HEADERS
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + SOURCES + ["-o", tmp]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
