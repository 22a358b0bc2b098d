"""Build libbgtq.so (the C-ABI library, include/bgtq.h) in-tree with nvcc for sm_100a.

``python -m paper_2606_24033_b200.build [--force] [--verbose]``; the result is
``paper_2606_24033_b200/libbgtq.so``.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libbgtq.so")
SOURCES = ["bgtq_host.cu", "bgtq_kernels.cu", "bgtq_append.cu", "bgtq_decode.cu", "bgtq_decode2.cu", "bgtq_microbench.cu", "codebook.cpp"]
HEADERS = ["bgtq_internal.h", "bgtq_device.cuh", os.path.join("..", "..", "include", "bgtq.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--compiler-options", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


OBJ = os.path.join(_HERE, "_obj")          # per-source objects (git-ignored): only stale sources are recompiled, in parallel


def _deps(src: str) -> list:
    return [os.path.join(CSRC, src)] + [os.path.join(CSRC, h) for h in HEADERS] + [os.path.abspath(__file__)]


def _obj(src: str) -> str:
    return os.path.join(OBJ, os.path.splitext(src)[0] + ".o")


def _stale(target: str, deps: list) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def needs_build() -> bool:
    return _stale(LIB, [d for s in SOURCES for d in _deps(s)])


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    from concurrent.futures import ThreadPoolExecutor
    os.makedirs(OBJ, exist_ok=True)
    extra = os.environ.get("BGTQ_EXTRA_NVCC", "").split()
    flags = [f for f in NVCC_FLAGS if f != "-shared"] + extra + (["-Xptxas", "-v"] if verbose else [])
    tag = os.path.join(OBJ, "flags.txt")        # objects built with other flags are stale
    if not os.path.exists(tag) or open(tag).read() != " ".join(flags):
        force = True

    def compile_one(src: str):
        if not force and not _stale(_obj(src), _deps(src)):
            return None
        return subprocess.run([_nvcc()] + flags + ["-c", src, "-o", _obj(src)], cwd=CSRC, capture_output=True, text=True)

    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as pool:
        results = list(pool.map(compile_one, SOURCES))
    failed = False
    for res in results:
        if res is not None and (verbose or res.returncode != 0):
            sys.stderr.write(res.stdout + res.stderr)
        failed |= res is not None and res.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed building libbgtq.so")
    with open(tag, "w") as f:
        f.write(" ".join(flags))
    res = subprocess.run([_nvcc(), "-shared", "-o", LIB] + [_obj(s) for s in SOURCES], cwd=CSRC, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed linking libbgtq.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
