"""Builds libidfx.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2304_13746_b200.build [--force] [-v]

Translation units: csrc/idfx.cu (C ABI, state kernels, fused CT/update kernel), csrc/probe.cu, and csrc/stage_inst.cu once
per (Riemann solver, reconstruction) pair, compiled in parallel as separate nvcc processes.  No -split-compile: with it
the code nvcc 12.9 generates for register-bound kernels (where their loads are scheduled, hence 0 to 96 bytes
of spills) was found in round 1 to change from one build of the same source to the next and with the core count of the build
machine (a 512^3 sweep then took 5.8 or 6.9 ms).  One process per unit is deterministic.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_OBJ = os.path.join(_HERE, "build")
SOURCES = [os.path.join(_CSRC, f) for f in ("idfx.cu", "probe.cu", "stage_inst.cu", "noalloc.cu")]
HEADERS = sorted(os.path.join(_CSRC, f) for f in os.listdir(_CSRC) if f.endswith(".cuh")) + [
    os.path.join(os.path.dirname(_HERE), "include", "idfx.h"), os.path.join(os.path.dirname(_HERE), "include", "idfx_probe.h"),
    os.path.join(os.path.dirname(_HERE), "include", "idfx_noalloc.h")]
LIB = os.path.join(_HERE, "libidfx.so")

# --register-usage-level=3 (default 5): ptxas keeps the fused CT/update kernel at 64 registers without its 16-32 B of spills
# (9.55 -> 9.1 ms at 512^3) and the sweeps at 150-168 registers with fewer spills (same speed)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "-Xfatbin", "-compress-all", "-Xptxas", "--register-usage-level=3"]
SOLVERS = (0, 1, 2, 3, 4)   # HLL, HLLC, HLLD, Roe, Rusanov (csrc/physics.cuh)
LIMITERS = (0, 1, 2, 3)     # flat, minmod, van Leer, LimO3


def _units(obj_dir):
    """(object path, nvcc arguments) of every translation unit, the longest first"""
    units = [(os.path.join(obj_dir, "idfx.o"), ["-c", SOURCES[0]])]
    for s in sorted(SOLVERS, key=lambda s: s != 3):   # Roe takes longest
        for l in reversed(LIMITERS):
            units.append((os.path.join(obj_dir, "stage_%d_%d.o" % (s, l)),
                          ["-DIDFX_INST_SOLVER=%d" % s, "-DIDFX_INST_LIM=%d" % l, "-c", SOURCES[2]]))
    units.append((os.path.join(obj_dir, "probe.o"), ["-c", SOURCES[1]]))
    units.append((os.path.join(obj_dir, "noalloc.o"), ["-c", SOURCES[3]]))
    return units


def build(force=False, verbose=False, extra_flags=(), lib=LIB, obj_dir=_OBJ):
    """extra_flags / lib / obj_dir: development builds of variants (-D switches) next to the product library"""
    deps = SOURCES + HEADERS + [os.path.abspath(__file__)]
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(d) for d in deps):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(obj_dir, exist_ok=True)
    units = _units(obj_dir)

    def compile_one(unit):
        obj, args = unit
        cmd = [nvcc] + NVCC_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) + args + ["-o", obj]
        subprocess.check_call(cmd)
        return obj

    workers = max(2, os.cpu_count() or 4)
    with ThreadPoolExecutor(max_workers=workers) as pool:
        objs = list(pool.map(compile_one, units))
    tmp = lib + ".tmp.%d" % os.getpid()
    subprocess.check_call([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"] + objs + ["-ldl", "-o", tmp])
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
