"""Build csrc/libkvpool.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2511_20982_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libkvpool.so")
SOURCES = ["kv_pool.cu"]
DEPS = SOURCES + ["kv_common.cuh", "kv_copy.cuh", "kv_attn.cuh", "kv_attn_tc.cuh", "kv_host.h", os.path.join("..", "..", "include", "kv_pool.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-Wall,-Wextra",
    "-shared", "-cudart", "static",
]


STAMP = LIB + ".srchash"


def source_hash() -> str:
    """sha256 over the sources, headers, flags and this file: what the built library must correspond to.
    (mtimes do not survive a copy of the tree to another box; contents do.)"""
    import hashlib
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for d in sorted(DEPS):
        with open(os.path.join(CSRC, d), "rb") as f:
            h.update(d.encode() + b"\0" + f.read())
    return h.hexdigest()


def stale() -> bool:
    """True if libkvpool.so is missing or was not built from the sources that are in the tree now."""
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = LIB + f".{os.getpid()}.tmp"
        cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp,
               *[os.path.join(CSRC, s) for s in SOURCES]]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
        os.replace(tmp, LIB)
        with open(STAMP, "w") as f:
            f.write(source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
