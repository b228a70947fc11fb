"""Build libmc_tvd.so (the C-ABI CUDA library, include/mc_tvd.h) in-tree with nvcc for sm_100a.

    python -m paper_2411_10372_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the tree to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

_PKG = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_PKG, "csrc")
LIB_PATH = os.path.join(_PKG, "libmc_tvd.so")
_SOURCES = ["mc_tvd.cu"]
_HASH_PATH = LIB_PATH + ".srchash"


def _deps() -> list[str]:
    """Every file the library is compiled from: all of csrc/ plus the public header."""
    files = sorted(os.path.join(_CSRC, f) for f in os.listdir(_CSRC) if f.endswith((".cu", ".cuh", ".h")))
    return files + [os.path.join(_PKG, "..", "include", "mc_tvd.h")]


NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _source_hash() -> str:
    """Content hash of the sources and flags (mtimes do not survive the copy to the GPU box)."""
    import hashlib
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for path in _deps():
        with open(path, "rb") as f:
            h.update(os.path.basename(path).encode() + b"\0" + f.read())
    return h.hexdigest()


def _stale() -> bool:
    if not (os.path.exists(LIB_PATH) and os.path.exists(_HASH_PATH)):
        return True
    with open(_HASH_PATH) as f:
        return f.read().strip() != _source_hash()


MAX_STACK_BYTES = 256


def _check_stack_frames(ptxas_log: str) -> None:
    """A sweep kernel whose march lambdas were not inlined keeps its register pipeline in local memory
    (seen once: 1472-byte frame, 6x slower).  ptxas -v reports the frame of every entry: refuse such a build."""
    import re
    entry = None
    for line in ptxas_log.splitlines():
        m = re.search(r"Compiling entry function '([^']+)'", line)
        if m:
            entry = m.group(1)
        m = re.search(r"(\d+) bytes stack frame", line)
        if m and entry and int(m.group(1)) > MAX_STACK_BYTES:
            raise RuntimeError(f"kernel {entry} has a {m.group(1)}-byte stack frame (> {MAX_STACK_BYTES}): "
                               "a lambda was not inlined or the register budget is too small")


def build_library(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale()):
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB_PATH + f".tmp{os.getpid()}"
    cmd = [nvcc] + NVCC_FLAGS + ["-o", tmp] + [os.path.join(_CSRC, s) for s in _SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(_PKG, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        sys.stderr.write(log)
        raise RuntimeError("nvcc failed building libmc_tvd.so")
    _check_stack_frames(log)
    os.replace(tmp, LIB_PATH)
    with open(_HASH_PATH, "w") as f:
        f.write(_source_hash() + "\n")
    if verbose:
        print(log)
    return LIB_PATH


if __name__ == "__main__":
    build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(LIB_PATH)
