"""Build liblsms_tau.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

Every csrc/*.cu is compiled to an object under build/ and the objects are linked into the shared library.
Staleness is decided by CONTENT (a hash of the sources, headers and flags stored beside each artefact), not by
mtimes, so a snapshot copied to another machine is not rebuilt for nothing and an edited source always is.
Concurrent callers (torchrun ranks on a fresh checkout) are serialised by a file lock; the library is written to a
temporary name and moved into place, so no process ever loads a half-written file.
"""
from __future__ import annotations

import fcntl
import glob
import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "liblsms_tau.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"] + os.environ.get("LSMS_NVCC_EXTRA", "").split()
LINK_FLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) +
                  glob.glob(os.path.join(INCLUDE, "*.h")))


def _digest(paths: list[str], extra: str = "") -> str:
    h = hashlib.sha256(extra.encode())
    for p in paths:
        h.update(os.path.basename(p).encode())
        with open(p, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def _stamp(path: str) -> str:
    try:
        with open(path + ".srchash") as f:
            return f.read().strip()
    except OSError:
        return ""


def lib_digest() -> str:
    return _digest(sources() + _headers(), " ".join(NVCC_FLAGS + LINK_FLAGS))


def needs_build() -> bool:
    return not os.path.exists(LIB) or _stamp(LIB) != lib_digest()


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    with open(os.path.join(OBJ, ".lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not (force or needs_build()):          # another process built it while we waited
            return LIB
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        hdrs = _headers()
        flags = NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else [])

        def compile_one(src: str) -> str:
            obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
            dig = _digest([src] + hdrs, " ".join(NVCC_FLAGS))
            if force or verbose or not os.path.exists(obj) or _stamp(obj) != dig:
                subprocess.check_call([nvcc] + flags + ["-c", "-o", obj, src])
                with open(obj + ".srchash", "w") as f:
                    f.write(dig)
            return obj

        with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
            objs = list(ex.map(compile_one, sources()))
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([nvcc] + LINK_FLAGS + ["-o", tmp] + objs)
        os.replace(tmp, LIB)
        with open(LIB + ".srchash", "w") as f:
            f.write(lib_digest())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
