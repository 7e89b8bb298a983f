"""Builds the C-ABI library `libllx.so` in-tree with nvcc for sm_100a (no JIT cache, no fallback)."""
from __future__ import annotations

import os
import shutil
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libllx.so")
SOURCES = [os.path.join(CSRC, "llx_api.cu"), os.path.join(CSRC, "llx_coord.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("llx_copy.cuh", "llx_attention.cuh", "llx_internal.h")] + \
    [os.path.join(os.path.dirname(HERE), "include", "llx.h")]

# -cudart shared: the library uses the process's CUDA runtime (the one torch already loaded, else the toolkit's through
# the rpath) instead of carrying a private static copy — one runtime per process, and the artefact holds our code only.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-diag-suppress", "550", "-cudart", "shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the llx library has no prebuilt or CPU fallback")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS if os.path.exists(d))


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libllx.so if missing or older than its sources; returns its path."""
    if not force and not is_stale():
        return LIB
    nvcc = _nvcc()
    cuda_lib = os.path.join(os.path.dirname(os.path.dirname(os.path.realpath(nvcc))), "lib64")
    cmd = [nvcc] + NVCC_FLAGS + ["-Xlinker", "-rpath=" + cuda_lib] + (["-Xptxas", "-v"] if verbose else []) + \
        ["-o", LIB + ".tmp"] + SOURCES
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    os.replace(LIB + ".tmp", LIB)
    if verbose:
        print(r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
