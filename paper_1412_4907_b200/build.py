"""Build libbf.so (CUDA kernels + C ABI) in-tree with nvcc for sm_100a.

    python -m paper_1412_4907_b200.build [--force] [-v] [--jitter]

Every csrc/*.cu is compiled to an object file of its own (in parallel, only when it or a header is newer than
the object), then linked into libbf.so.  --jitter builds libbf_jitter.so instead: the same sources with -DBF_JITTER=1
(random sleeps in front of every mbarrier wait, csrc/ptx.cuh) -- a TEST library for tests/test_zy_jitter.py, never
loaded unless BF_LIBRARY points at it.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libbf.so")

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def headers():
    return (glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh"))
            + [os.path.join(HERE, "..", "include", "bf.h")])


JITTER_OBJ = os.path.join(HERE, "build_jitter")
JITTER_LIB = os.path.join(HERE, "libbf_jitter.so")


def _obj(src: str, objdir: str = OBJ) -> str:
    return os.path.join(objdir, os.path.basename(src)[:-3] + ".o")


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def needs_build(jitter: bool = False) -> bool:
    return _stale(JITTER_LIB if jitter else LIB, sources() + headers())


def build(force: bool = False, verbose: bool = False, jitter: bool = False) -> str:
    lib, objdir = (JITTER_LIB, JITTER_OBJ) if jitter else (LIB, OBJ)
    if not (force or needs_build(jitter)):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(objdir, exist_ok=True)
    hdrs = headers()
    todo = [s for s in sources() if force or _stale(_obj(s, objdir), [s] + hdrs)]
    flags = NVCC_FLAGS + (["-DBF_JITTER=1"] if jitter else [])

    def compile_one(src: str) -> None:
        cmd = [nvcc] + flags + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", _obj(src, objdir), src]
        subprocess.run(cmd, check=True)

    with ThreadPoolExecutor(max_workers=min(len(todo), os.cpu_count() or 4) or 1) as pool:
        list(pool.map(compile_one, todo))
    # objects of sources that no longer exist must not be linked
    objs = [_obj(s, objdir) for s in sources()]
    subprocess.run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", lib] + objs, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, jitter="--jitter" in sys.argv))
