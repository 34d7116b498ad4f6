"""Build libjefi.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libjefi.so")
SOURCES = ["jefi_api.cu", "jefi_field.cu", "jefi_particles.cu", "jefi_probe.cu"]
HEADERS = [os.path.join(CSRC, "jefi_ctx.h"), os.path.join(ROOT, "include", "jefi.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(p) > t for p in deps)


LIB_CHECKED = os.path.join(HERE, "libjefi_checked.so")


def build_lib(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo ... -> paper_2209_07944_b200/libjefi.so
    checked=True builds libjefi_checked.so with -DJEFI_CHECKED: the same library with its own device-side memory checks
    (include/jefi.h, jefi_debug_check_errors); the GPU tests run against it when JEFI_LIBRARY points at it."""
    lib = LIB_CHECKED if checked else LIB
    if not force and not checked and not _stale():
        return lib
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-o", lib]
    if checked:
        cmd += ["-DJEFI_CHECKED"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv, checked="--checked" in sys.argv))
