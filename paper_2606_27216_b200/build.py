"""Build libhimuon.so (the C-ABI library of include/himuon.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_27216_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  Every .cu is compiled to its own object (in parallel, cached by a
fingerprint of the source, the headers and the flags) and the objects are linked into the shared object,
which lands next to this file so that it travels with the repository snapshot to the GPU box (it is
git-ignored).
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

PKG_DIR = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(PKG_DIR)
CSRC = os.path.join(PKG_DIR, "csrc")
OBJ_DIR = os.path.join(PKG_DIR, "build")
LIB_PATH = os.path.join(PKG_DIR, "libhimuon.so")
STAMP_PATH = os.path.join(PKG_DIR, "libhimuon.stamp")

SOURCES = sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))
HEADERS = sorted(f for f in os.listdir(CSRC) if f.endswith((".h", ".cuh"))) + [os.path.join(ROOT, "include", "himuon.h")]

COMPILE_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-Xcompiler", "-fPIC", "-ldl"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _read(path: str) -> bytes:
    with open(path, "rb") as fh:
        return fh.read()


def _header_hash() -> str:
    h = hashlib.sha256()
    for f in HEADERS:
        h.update(_read(f if os.path.isabs(f) else os.path.join(CSRC, f)))
    return h.hexdigest()


def _fingerprint(extra_flags=()) -> str:
    h = hashlib.sha256()
    for f in SOURCES:
        h.update(_read(os.path.join(CSRC, f)))
    h.update(_header_hash().encode())
    h.update(" ".join(COMPILE_FLAGS + LINK_FLAGS + list(extra_flags)).encode())
    return h.hexdigest()


def _compile_one(src: str, obj_dir: str, hdr: str, extra_flags, force: bool, verbose: bool):
    """Compile csrc/<src> -> <obj_dir>/<src>.o unless its fingerprint is unchanged; returns (obj, log)."""
    obj = os.path.join(obj_dir, src + ".o")
    stamp = obj + ".stamp"
    h = hashlib.sha256(_read(os.path.join(CSRC, src)))
    h.update(hdr.encode())
    h.update(" ".join(COMPILE_FLAGS + list(extra_flags)).encode())
    fp = h.hexdigest()
    if not force and os.path.exists(obj) and os.path.exists(stamp) and _read(stamp).decode().strip() == fp:
        return obj, ""
    cmd = [_nvcc()] + COMPILE_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) + \
          ["-c", os.path.join(CSRC, src), "-o", obj]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}:\n{res.stdout}{res.stderr}")
    with open(stamp, "w") as fh:
        fh.write(fp)
    return obj, res.stdout + res.stderr


def build(force: bool = False, verbose: bool = False, extra_flags=(), lib_path: str = LIB_PATH,
          obj_dir: str = OBJ_DIR) -> str:
    """Compile what changed, link, and return the path of the shared library.

    `extra_flags` / `lib_path` / `obj_dir` let a development build (e.g. -DHIMUON_TRACE) live beside the product
    library without touching it."""
    stamp_path = STAMP_PATH if lib_path == LIB_PATH else lib_path + ".stamp"
    fp = _fingerprint(extra_flags)
    if not force and os.path.exists(lib_path) and os.path.exists(stamp_path):
        if _read(stamp_path).decode().strip() == fp:
            return lib_path
    os.makedirs(obj_dir, exist_ok=True)
    hdr = _header_hash()
    with ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 4)) as pool:
        results = list(pool.map(lambda s: _compile_one(s, obj_dir, hdr, extra_flags, force, verbose), SOURCES))
    if verbose:
        for _, log in results:
            sys.stderr.write(log)
    cmd = [_nvcc()] + LINK_FLAGS + [o for o, _ in results] + ["-o", lib_path]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed linking libhimuon.so (see stderr)")
    with open(stamp_path, "w") as fh:
        fh.write(fp)
    return lib_path


DEBUG_LIB_PATH = os.path.join(PKG_DIR, "libhimuon_debug.so")


def build_debug(force: bool = False, verbose: bool = False) -> str:
    """The -DHIMUON_DEBUG_STAGES build: same sources plus the accumulator-dump stages of the T = 128 kernels and their
    `himuon_debug_set_*` exports.  Only the stage tests load it; the product library has none of this."""
    return build(force=force, verbose=verbose, extra_flags=("-DHIMUON_DEBUG_STAGES",), lib_path=DEBUG_LIB_PATH,
                 obj_dir=os.path.join(PKG_DIR, "build_debug"))


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    if "--debug" in sys.argv:
        print(build_debug(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
