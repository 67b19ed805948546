"""Build libhimuon.so (the C-ABI library of include/himuon.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_27216_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The shared object lands next to this file so that it travels
with the repository snapshot to the GPU box (it is git-ignored).
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG_DIR)
CSRC = os.path.join(PKG_DIR, "csrc")
LIB_PATH = os.path.join(PKG_DIR, "libhimuon.so")
STAMP_PATH = os.path.join(PKG_DIR, "libhimuon.stamp")

SOURCES = ["himuon_api.cu", "kernels_simt.cu", "kernels_tc128.cu", "kernels_tc128_fp8.cu", "kernels_tc64.cu", "kernels_tc256.cu", "kernels_tc256_fp8.cu", "kernels_warp.cu", "kernels_gemm.cu"]
HEADERS = ["himuon_internal.h", "sm100_ptx.cuh", "tc_common.cuh", os.path.join(ROOT, "include", "himuon.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-ldl",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _fingerprint() -> str:
    h = hashlib.sha256()
    for f in SOURCES + HEADERS:
        p = f if os.path.isabs(f) else os.path.join(CSRC, f)
        with open(p, "rb") as fh:
            h.update(fh.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if sources changed; return the path of the shared library."""
    fp = _fingerprint()
    if not force and os.path.exists(LIB_PATH) and os.path.exists(STAMP_PATH):
        with open(STAMP_PATH) as fh:
            if fh.read().strip() == fp:
                return LIB_PATH
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB_PATH]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libhimuon.so (see stderr)")
    with open(STAMP_PATH, "w") as fh:
        fh.write(fp)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
