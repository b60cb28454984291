"""Compile the CUDA library paper_1412_6367_b200/libazint.so for sm_100a with nvcc (in-tree, no JIT cache).

Every .cu of csrc/ is compiled to an object file under csrc/.obj/ (in parallel, only when it or a header changed),
then the objects are linked into the shared library.

Usage: python -m paper_1412_6367_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, ".obj")
LIB = os.path.join(HERE, "libazint.so")
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-O2,-Wall",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "--shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        [os.path.join(os.path.dirname(HERE), "include", "azint.h")]


def _mtime(path):
    return os.path.getmtime(path) if os.path.exists(path) else -1.0


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib_path: str = LIB) -> str:
    """Returns the path of the library; recompiles only what is older than its source or any header."""
    nvcc = os.environ.get("NVCC", "nvcc")
    obj_dir = OBJ if lib_path == LIB else lib_path + ".obj"
    os.makedirs(obj_dir, exist_ok=True)
    hdr_time = max(_mtime(h) for h in _headers())
    jobs = []
    for src in sources():
        obj = os.path.join(obj_dir, os.path.basename(src)[:-3] + ".o")
        if force or _mtime(obj) < max(_mtime(src), hdr_time):
            jobs.append((src, obj))
    objs = [os.path.join(obj_dir, os.path.basename(s)[:-3] + ".o") for s in sources()]
    if not jobs and _mtime(lib_path) >= max(_mtime(o) for o in objs):
        return lib_path

    def compile_one(job):
        src, obj = job
        tmp = obj + f".tmp{os.getpid()}"
        cmd = [nvcc, *NVCC_FLAGS, *extra_flags, *(["-Xptxas", "-v"] if verbose else []), "-c", src, "-o", tmp]
        subprocess.check_call(cmd)
        os.replace(tmp, obj)

    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as pool:
            list(pool.map(compile_one, jobs))
    tmp = lib_path + f".tmp{os.getpid()}"
    subprocess.check_call([nvcc, *LINK_FLAGS, *objs, "-o", tmp])
    os.replace(tmp, lib_path)
    return lib_path


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
