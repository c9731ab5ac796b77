"""Build libsparrow_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libsparrow_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-diag-suppress", "550", "-Xcompiler", "-fPIC", "-shared"]


def sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))) + [
        os.path.join(_HERE, "..", "include", "sparrow.h")]


def source_hash() -> str:
    """Short hash of the kernel sources + the C header: names the build a measurement (e.g. an ncu capture) was taken on.
    Comments and whitespace are left out of it, so a documentation edit does not orphan the captures under profiles/."""
    import hashlib
    import re
    h = hashlib.sha256()
    for f in sources():
        h.update(os.path.basename(f).encode())
        text = open(f, "r", encoding="utf-8").read()
        text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)          # block comments
        text = re.sub(r"(?<![:\"'])//[^\n]*", " ", text)            # line comments (not the // of a string or URL)
        h.update(" ".join(text.split()).encode())
    return h.hexdigest()[:12]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


LIB_TRACE = os.path.join(_HERE, "libsparrow_b200_trace.so")


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    """trace=True: the tracing build (-DSPARROW_TRACE, csrc/common.cuh) beside the normal one; loaded through
    SPARROW_B200_LIB (binding.py), used by trace.py."""
    lib = LIB_TRACE if trace else LIB
    if force or trace or stale():
        cmd = [NVCC, *FLAGS, *(["-DSPARROW_TRACE"] if trace else []), *(["-Xptxas", "-v"] if verbose else []), "-o", lib,
               os.path.join(CSRC, "api.cu")]
        subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
