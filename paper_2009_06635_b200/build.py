"""Build libpdfb200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpdfb200.so")
PROBE_LIB = os.path.join(HERE, "libpdfb200_probe.so")  # bench utility, a library of its own (include/pdfb200_probe.h)
PROBE_SRC = os.path.join(CSRC, "probe", "probes.cu")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC,-O2,-Wall", "--shared", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(PROBE_LIB))
    deps = sources() + [PROBE_SRC] + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(HERE, "..", "include", "*.h")) + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        extra = os.environ.get("PDFB_BUILD_FLAGS", "").split()  # e.g. -DPDFB_CHECKED: the bounds-checked build
        for lib, srcs in ((LIB, sources()), (PROBE_LIB, [PROBE_SRC])):
            cmd = [NVCC] + FLAGS + extra + ["-o", lib] + srcs
            res = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or res.returncode != 0:
                sys.stderr.write(res.stdout + res.stderr)
            if res.returncode != 0:
                raise RuntimeError("nvcc failed building " + os.path.basename(lib))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
