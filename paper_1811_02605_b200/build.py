"""Builds csrc/mas_pcg.cu for sm_100a, in-tree (so the .so files travel with gpurun):

    lib/libmas_pcg.so      the product library (include/mas_pcg.h)
    lib/libmas_pcg_dbg.so  the same source with -DMAS_PCG_DEBUG_PROBES: adds the measurement probes of
                           include/mas_pcg_debug.h (per-kernel CUDA-event timing, traffic-mix probe) for bench.py

    python -m paper_1811_02605_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "lib", "libmas_pcg.so")
LIB_DBG = os.path.join(_HERE, "lib", "libmas_pcg_dbg.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh"))
                  + glob.glob(os.path.join(CSRC, "*.inc")) + glob.glob(os.path.join(INCLUDE, "*.h")))


def up_to_date() -> bool:
    for lib in (LIB, LIB_DBG):
        if not os.path.exists(lib):
            return False
        t = os.path.getmtime(lib)
        if not all(os.path.getmtime(s) <= t for s in sources()):
            return False
    return True


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(os.path.dirname(LIB), exist_ok=True)
    jobs = []
    for lib, extra in ((LIB, []), (LIB_DBG, ["-DMAS_PCG_DEBUG_PROBES"])):
        tmp = f"{lib}.{os.getpid()}.tmp"
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-o", tmp, os.path.join(CSRC, "mas_pcg.cu")]
        jobs.append((lib, tmp, cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)))
    logs = []
    for lib, tmp, cmd, proc in jobs:
        out, err = proc.communicate()
        if proc.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + out + err)
        os.replace(tmp, lib)
        logs.append(" ".join(cmd) + "\n" + err)
    with open(os.path.join(os.path.dirname(LIB), "ptxas.log"), "w") as f:
        f.write(logs[0])
    if verbose:
        print(logs[0])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
