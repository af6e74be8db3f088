"""Builds libcacheweaver.so (C ABI, include/cacheweaver.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_19667_b200.build [--force]
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

PKG = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG)
CSRC = os.path.join(PKG, "csrc")
LIB = os.path.join(PKG, "libcacheweaver.so")
STAMP = LIB + ".srchash"          # hash of the sources + flags the library was built from (written next to it)
SOURCES = ["host.cpp", "append_kv.cu", "prefill_attn.cu", "api.cu"]
HEADERS = ["cw_internal.h", "ptx_sm100.cuh", os.path.join(ROOT, "include", "cacheweaver.h")]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def _flags() -> list:
    return ["-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler",
            "-fPIC,-Wall,-Wno-unused-function"]


def source_hash() -> str:
    """sha256 over the build flags and the contents of every source and header (file names included)."""
    h = hashlib.sha256(" ".join(_flags()).encode())
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [x if os.path.isabs(x) else os.path.join(CSRC, x) for x in HEADERS]
    for d in deps:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def _stale() -> bool:
    """The library is current iff its stamp file holds the hash of today's sources (mtimes are meaningless after a
    clone or an rsync)."""
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as f:
        return f.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    cmd = [_nvcc()] + _flags() + ["-I", os.path.join(ROOT, "include"), "-I", CSRC, "-x", "cu"] + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    with open(STAMP, "w") as f:
        f.write(source_hash() + "\n")
    if verbose:
        print(r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
