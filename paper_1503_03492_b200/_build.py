"""Build libsmre.so (C ABI of include/smre.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libsmre.so")
SOURCES = ["smre_api.cu", "smre_family.cu", "smre_icd.cu", "smre_conveyor.cu", "smre_conveyor_plan.cu", "smre_strips.cu", "smre_noalloc.cu", "smre_calibrate.cu", "smre_admm.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    deps.append(os.path.join(os.path.dirname(_HERE), "include", "smre.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, *NVCC_FLAGS, "-o", LIB, *[os.path.join(CSRC, s) for s in SOURCES]]
        if os.environ.get("SMRE_CV_TRACE_BUILD"):
            cmd.insert(1, "-DSMRE_CV_TRACE_BUILD=" + os.environ["SMRE_CV_TRACE_BUILD"])
        if os.environ.get("SMRE_ST_KO_BUILD"):
            cmd.insert(1, "-DSMRE_ST_KO")
        if os.environ.get("SMRE_DEBUG"):
            cmd.insert(1, "-DSMRE_DEBUG")
        else:
            cmd.insert(1, "-DNDEBUG")
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd))
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
