"""Build librmsynth.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_1810_06250_b200.build [--force] [-v] [--timeline]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box, so "is it up to
date" is decided by CONTENT, not by mtimes: a SHA-256 over csrc/*, include/rmsynth.h and the compiler flags
is compiled into the library (rmsynth_version() reports it) and written next to it; build() recompiles
whenever the hash of the sources on disk differs from the one the binary was built from.

--timeline builds librmsynth_timeline.so, the same sources with -DRMSYNTH_TIMELINE (per-role clock64
stamps in the FP16 tensor kernel, read back through rmsynth_timeline_read).  Debug only.
"""
from __future__ import annotations

import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librmsynth.so")
LIB_TIMELINE = os.path.join(HERE, "librmsynth_timeline.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC,-O2", "-I", os.path.join(ROOT, "include"), "-I", CSRC]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def source_hash(extra=()) -> str:
    """SHA-256 (first 16 hex digits) of every file the library is compiled from, plus the flags."""
    h = hashlib.sha256()
    deps = sources() + sorted(glob.glob(os.path.join(CSRC, "*.cuh"))) + [os.path.join(ROOT, "include", "rmsynth.h")]
    for d in deps:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    h.update(" ".join(FLAGS[:8] + list(extra)).encode())
    return h.hexdigest()[:16]


def built_hash(lib: str) -> str | None:
    try:
        with open(lib + ".hash") as f:
            return f.read().strip()
    except OSError:
        return None


def stale(lib: str = LIB, extra=()) -> bool:
    return not os.path.exists(lib) or built_hash(lib) != source_hash(extra)


def build(force: bool = False, verbose: bool = False, timeline: bool = False) -> str:
    lib = LIB_TIMELINE if timeline else LIB
    extra = ["-DRMSYNTH_TIMELINE"] if timeline else []
    if not (force or stale(lib, extra)):
        return lib
    digest = source_hash(extra)
    objdir = os.path.join(HERE, "build", "timeline" if timeline else "product")
    os.makedirs(objdir, exist_ok=True)
    objs, procs = [], []
    for src in sources():
        obj = os.path.join(objdir, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        cmd = [NVCC, *FLAGS, *extra, f'-DRMSYNTH_SOURCE_HASH="{digest}"', "-c", src, "-o", obj] + (["-Xptxas", "-v"] if verbose else [])
        procs.append((cmd, subprocess.Popen(cmd)))
    for cmd, pr in procs:
        if pr.wait() != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    cmd = [NVCC, "-shared", "-o", lib, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static"]
    subprocess.run(cmd, check=True)
    with open(lib + ".hash", "w") as f:
        f.write(digest + "\n")
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, timeline="--timeline" in sys.argv))
