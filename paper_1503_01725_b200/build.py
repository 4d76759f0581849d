"""Builds libpslmc.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1503_01725_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpslmc.so")
SOURCES = ["pslmc_psl.cu", "pslmc_dose.cu", "pslmc_static.cu"]
PROBE_LIB = os.path.join(HERE, "libpslmc_probe.so")           # measurement probes (probes.py), not part of the ABI
PROBE_SOURCES = [os.path.join("probes", "mem_probe.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
              "-shared", "-Xcompiler", "-fPIC"]


def _stale(lib: str, deps: list) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    core = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if os.path.isfile(os.path.join(CSRC, f))] + [os.path.join(HERE, "..", "include", "pslmc.h")]
    for lib, sources, deps in ((LIB, SOURCES, core), (PROBE_LIB, PROBE_SOURCES, [os.path.join(CSRC, s) for s in PROBE_SOURCES])):
        if force or _stale(lib, deps):
            tmp = lib + ".tmp%d" % os.getpid()
            cmd = [nvcc] + NVCC_FLAGS + os.environ.get("PSLMC_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, s) for s in sources]
            subprocess.check_call(cmd)
            os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
