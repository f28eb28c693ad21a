"""Build libng.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libng.so")
SOURCES = [os.path.join(CSRC, "ng.cu"), os.path.join(CSRC, "ng_noalloc.cu")]
HEADERS = [os.path.join(CSRC, "ng_device.cuh"), os.path.join(os.path.dirname(_HERE), "include", "ng.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-DNG_EVICT_HINTS=2",
              "-shared", "-Xcompiler", "-fPIC"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ng.cu + csrc/ng_noalloc.cu -> libng.so if missing or older than its sources.  Raises if nvcc fails.
    NG_LIB=<path> makes the binding load that prebuilt library instead (kernel experiments built with other flags)."""
    if os.environ.get("NG_LIB"):
        return os.environ["NG_LIB"]
    if force or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + SOURCES + ["-o", LIB]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build_lib(force=True, verbose=True))
