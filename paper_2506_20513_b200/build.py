"""Build libgprfwi.so in-tree with nvcc for sm_100a (`python -m paper_2506_20513_b200.build`)."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libgprfwi.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--use_fast_math=false", "-Xcompiler", "-fPIC", "-shared"]


def _sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh")))


def build(force: bool = False, verbose: bool = False) -> str:
    deps = _sources() + [os.path.join(_ROOT, "include", "gprfwi.h")]
    if (not force and os.path.exists(LIB_PATH)
            and os.path.getmtime(LIB_PATH) >= max(os.path.getmtime(d) for d in deps)):
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    flags += os.environ.get("GPRFWI_NVCC_EXTRA", "").split()       # tuning builds, e.g. -DGPRFWI_PROBE
    tmp = LIB_PATH + f".tmp{os.getpid()}"
    cmd = [nvcc, *flags, *(["-Xptxas", "-v"] if verbose else []), "-I", os.path.join(_ROOT, "include"),
           "-I", CSRC, "-o", tmp, os.path.join(CSRC, "gprfwi.cu")]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
