"""Build libpsfft.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1808_01309_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the repo snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libpsfft.so")
SOURCES = ["psfft_api.cu"] + [f"psfft_{dt}_{grp}.cu" for dt in ("f64", "f32") for grp in ("midx", "colc", "cola", "fft")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", INCLUDE]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    return "nvcc"


def _flags(extra=()) -> str:
    return " ".join(NVCC_FLAGS[:6] + list(extra))


def _stamp() -> str:
    return os.path.join(HERE, "build", "flags.txt")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    # a library built with other flags (e.g. a size-restricted experimental build) is stale
    if not os.path.exists(_stamp()) or open(_stamp()).read() != _flags():
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "psfft.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    """Compile the translation units in parallel and link libpsfft.so.  Returns its path.
    extra_flags: additional nvcc flags of a development build (recorded in the stamp, so the next plain call
    rebuilds the product library); the product is always built with NVCC_FLAGS alone."""
    if not force and not _stale():
        return LIB
    nvcc = _nvcc()
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    extra = ["-Xptxas", "-v"] if verbose else []
    extra += list(extra_flags)

    # an object is reused when it was built with the same flags and is newer than everything its unit includes:
    # its own .cu, every .cuh, and (the boundary unit only) include/psfft.h
    same_flags = not force and os.path.exists(_stamp()) and open(_stamp()).read() == _flags(extra_flags)
    headers = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith(".cuh")]

    def compile_one(src: str) -> str:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        deps = [os.path.join(CSRC, src), *headers] + ([os.path.join(INCLUDE, "psfft.h")] if src == "psfft_api.cu" else [])
        if same_flags and not verbose and os.path.exists(obj) and all(os.path.getmtime(d) < os.path.getmtime(obj) for d in deps):
            return obj
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.check_call([nvcc, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    with open(_stamp(), "w") as f:
        f.write(_flags(extra_flags))
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
