"""Builds libnbody_b200.so (in-tree) from csrc/ with nvcc for sm_100a.  No JIT cache, no torch extension."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnbody_b200.so")
SOURCES = ["nbody_b200.cu", "nb_small_launch.cu", "nb_small_hermite_launch.cu"]
DEPS = ["nbody_b200.cu", "nb_small_launch.cu", "nb_small_launch.h", "nb_small.cuh", "nb_small_hermite_launch.cu", "nb_small_hermite_launch.h", "nb_small_hermite.cuh", "nb_hermite_pair.cuh", os.path.join(ROOT, "include", "nb_packed.cuh"), os.path.join(ROOT, "include", "nb_debug.h"), "nb_kernels.cuh", "nb_hermite.cuh", "nb_batched.cuh", "nb_pipelines.cuh", os.path.join(ROOT, "include", "nb_pipeline.cuh"), "nb_plan.h", os.path.join(ROOT, "include", "nbody_b200.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-I", os.path.join(ROOT, "include"),
]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    for d in DEPS:
        p = d if os.path.isabs(d) else os.path.join(CSRC, d)
        if os.path.getmtime(p) > t:
            return True
    return False


def build(force: bool = False, verbose: bool = False) -> str:
    """One object per translation unit, compiled side by side, then one shared library."""
    if force or stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        objs, procs = [], []
        for src in SOURCES:
            obj = os.path.join(CSRC, src.replace(".cu", ".o"))
            cmd = [nvcc, *NVCC_FLAGS, "-c", "-o", obj, os.path.join(CSRC, src)]
            if verbose:
                cmd[1:1] = ["-Xptxas", "-v"]
                print(" ".join(cmd), file=sys.stderr)
            objs.append(obj)
            procs.append((cmd, subprocess.Popen(cmd)))
        for cmd, p in procs:
            if p.wait() != 0:
                raise subprocess.CalledProcessError(p.returncode, cmd)
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB + ".tmp", *objs], check=True)
        os.replace(LIB + ".tmp", LIB)
        for obj in objs:
            os.remove(obj)
    return LIB


def build_microloops() -> str:
    """The stand-alone micro-benchmarks behind the roofline peak (csrc/nb_microloops.cu) -> nb_microloops (in-tree)."""
    out = os.path.join(HERE, "nb_microloops")
    nvcc = os.environ.get("NVCC", "nvcc")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-o", out,
                    os.path.join(CSRC, "nb_microloops.cu")], check=True)
    return out


if __name__ == "__main__":
    if "--microloops" in sys.argv:
        print(build_microloops())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
