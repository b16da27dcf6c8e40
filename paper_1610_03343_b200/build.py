"""Build the C-ABI library libmd_b200.so in-tree with nvcc for sm_100a (no JIT cache).

Every csrc/*.cu is compiled to an object under csrc/build/ (in parallel, only the stale ones) and the objects are
linked into the shared library.  The library is written to a temporary name and renamed, under a file lock, so
that several processes (torchrun ranks) asking for a stale library at once do not write into each other's output.
"""
from __future__ import annotations

import fcntl
import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

_DIR = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_DIR, "csrc")
OBJ = os.path.join(CSRC, "build")
INCLUDE = os.path.join(os.path.dirname(_DIR), "include")
LIB = os.path.join(_DIR, "libmd_b200.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def headers():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(INCLUDE, "md.h")]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in sources() + headers())


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or stale()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("MD_NVCC_EXTRA", "").split()       # e.g. -DMD_SW_MAXREG=168 for an A/B build
    os.makedirs(OBJ, exist_ok=True)
    with open(os.path.join(OBJ, ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not (force or stale()):                            # another process built it while we waited
            return LIB
        hdr_t = max(os.path.getmtime(h) for h in headers())
        flags = NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else [])
        stamp = os.path.join(OBJ, ".flags")
        same_flags = os.path.exists(stamp) and open(stamp).read() == " ".join(flags)

        def compile_one(src):
            obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
            if (not force and same_flags and os.path.exists(obj)
                    and os.path.getmtime(obj) > max(hdr_t, os.path.getmtime(src))):
                return obj
            subprocess.check_call([nvcc] + flags + ["-I", INCLUDE, "-I", CSRC, "-c", src, "-o", obj])
            return obj

        with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
            objs = list(pool.map(compile_one, sources()))
        open(stamp, "w").write(" ".join(flags))
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
