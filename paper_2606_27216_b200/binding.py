"""Thin ctypes binding of the C-ABI in include/himuon.h (same names, argument marshalling only).

Every step of the hot path runs inside libhimuon.so's CUDA kernels; this module only turns torch
tensors into {ptr, H, W, ld, dtype} descriptors and checks status codes.  There is no CPU or
PyTorch fallback: if the shared library is missing, loading raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np
import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libhimuon.so")

HIMUON_OK = 0
HIMUON_ERR_INVALID_ARG = 1
HIMUON_ERR_UNSUPPORTED = 2
HIMUON_ERR_WORKSPACE_TOO_SMALL = 3
HIMUON_ERR_CUDA = 4
HIMUON_ERR_NOT_BOUND = 5

HIMUON_F32, HIMUON_BF16 = 0, 1
HIMUON_PATH_AUTO, HIMUON_PATH_FP32, HIMUON_PATH_FP8 = 0, 1, 2

# PAPER.md:74 Eq. (2.3)
NS_COEFFS = (3.4445, -4.7750, 2.0315)


class himuon_mat(C.Structure):
    _fields_ = [("ptr", C.c_void_p), ("H", C.c_int32), ("W", C.c_int32), ("ld", C.c_int64),
                ("dtype", C.c_int32)]


class himuon_layer(C.Structure):
    _fields_ = [("w", himuon_mat), ("g", himuon_mat), ("m", himuon_mat), ("T", C.c_int32), ("T_w", C.c_int32)]


class himuon_hparams(C.Structure):
    _fields_ = [("K", C.c_int32), ("a", C.c_float), ("b", C.c_float), ("c", C.c_float),
                ("eps", C.c_float), ("beta", C.c_float), ("nesterov", C.c_int32),
                ("lr", C.c_float), ("wd", C.c_float), ("scale_c", C.c_float)]


class HimuonError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        lib = _lib()
        name = lib.himuon_status_string(status).decode()
        detail = lib.himuon_last_cuda_error().decode() if status == HIMUON_ERR_CUDA else ""
        super().__init__(f"{where}: {name}" + (f" ({detail})" if detail else ""))


_LIB = None
_LIBS = {}


def _load(path: str):
    """dlopen `path` and declare the C-ABI of include/himuon.h on it."""
    if path in _LIBS:
        return _LIBS[path]
    if not os.path.exists(path):
        raise ImportError(
            f"{path} not found: build it with `python -m paper_2606_27216_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(path)
    P = C.POINTER
    lib.himuon_plan_create.restype = C.c_int
    lib.himuon_plan_create.argtypes = [P(himuon_layer), C.c_int32, C.c_int32, C.c_int32, C.c_size_t,
                                       P(C.c_void_p)]
    lib.himuon_plan_info.restype = C.c_int
    lib.himuon_plan_info.argtypes = [C.c_void_p, P(C.c_int64), P(C.c_int32), P(C.c_int32), P(C.c_size_t)]
    lib.himuon_plan_worklist.restype = C.c_int
    lib.himuon_plan_worklist.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.himuon_plan_chunks.restype = C.c_int
    lib.himuon_plan_chunks.argtypes = [C.c_int64, C.c_int64, C.c_int64, C.c_int64, P(C.c_int32),
                                       C.c_void_p, C.c_int32]
    lib.himuon_plan_bind.restype = C.c_int
    lib.himuon_plan_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
    lib.himuon_plan_destroy.restype = None
    lib.himuon_plan_destroy.argtypes = [C.c_void_p]
    lib.himuon_step.restype = C.c_int
    lib.himuon_step.argtypes = [C.c_void_p, P(himuon_hparams), C.c_void_p]
    lib.himuon_phi.restype = C.c_int
    lib.himuon_phi.argtypes = [C.c_void_p, P(himuon_hparams), C.c_void_p]
    lib.himuon_ns_tiles.restype = C.c_int
    lib.himuon_ns_tiles.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_int32,
                                    C.c_int32, C.c_float, C.c_float, C.c_float, C.c_float,
                                    C.c_void_p, C.c_size_t, C.c_void_p]
    lib.himuon_ns_tiles_workspace_bytes.restype = C.c_size_t
    lib.himuon_ns_tiles_workspace_bytes.argtypes = []
    lib.himuon_ns_tiles_static.restype = C.c_int
    lib.himuon_ns_tiles_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32,
                                           C.c_float, C.c_float, C.c_float, C.c_float, C.c_void_p]
    lib.himuon_ns_tiles_static_max_tiles.restype = C.c_int64
    lib.himuon_ns_tiles_static_max_tiles.argtypes = [C.c_int32]
    lib.himuon_status_string.restype = C.c_char_p
    lib.himuon_status_string.argtypes = [C.c_int]
    lib.himuon_last_cuda_error.restype = C.c_char_p
    lib.himuon_last_cuda_error.argtypes = []
    lib.himuon_supported_tile_sizes.restype = C.c_int32
    lib.himuon_supported_tile_sizes.argtypes = [C.c_int32, C.c_int32]
    lib.himuon_launch_count.restype = C.c_int64
    lib.himuon_launch_count.argtypes = []
    _LIBS[path] = lib
    return lib


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = _load(LIB_PATH)
    return _LIB


class use_library:
    """Context manager: route the binding to another build of the same C-ABI (the -DHIMUON_DEBUG_STAGES library of
    the stage tests).  Plans created inside must be destroyed inside."""

    def __init__(self, path: str):
        self.path = path

    def __enter__(self):
        global _LIB
        self.prev = _LIB
        _LIB = _load(self.path)
        return _LIB

    def __exit__(self, *exc):
        global _LIB
        _LIB = self.prev
        return False


def _check(status: int, where: str):
    if status != HIMUON_OK:
        raise HimuonError(status, where)


def _dtype_code(dt: torch.dtype) -> int:
    if dt == torch.float32:
        return HIMUON_F32
    if dt == torch.bfloat16:
        return HIMUON_BF16
    raise TypeError(f"unsupported storage dtype {dt}")


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        if torch.cuda.is_available():
            return torch.cuda.current_stream().cuda_stream or None
        return None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


def mat_of(t: Optional[torch.Tensor]) -> himuon_mat:
    """{ptr, H, W, ld, dtype} of a 2-D row-major tensor (stride(1) == 1)."""
    if t is None:
        return himuon_mat(None, 0, 0, 0, 0)
    if t.dim() != 2 or (t.shape[1] > 1 and t.stride(1) != 1):
        raise ValueError("expected a 2-D tensor with unit column stride")
    ld = t.stride(0) if t.shape[0] > 1 else max(t.stride(0), t.shape[1])
    return himuon_mat(t.data_ptr(), t.shape[0], t.shape[1], ld, _dtype_code(t.dtype))


def shape_mat(H: int, W: int, dtype_code: int = HIMUON_BF16, ld: Optional[int] = None) -> himuon_mat:
    """Descriptor with a NULL pointer (plan inspection without device memory)."""
    return himuon_mat(None, H, W, W if ld is None else ld, dtype_code)


@dataclass
class HParams:
    """Hyper-parameters of Algorithm 4.1 (defaults)."""
    K: int = 5
    a: float = NS_COEFFS[0]
    b: float = NS_COEFFS[1]
    c: float = NS_COEFFS[2]
    eps: float = 1e-7
    beta: float = 0.95
    nesterov: bool = True
    lr: float = 0.02
    wd: float = 0.0
    scale_c: float = 0.2

    def to_c(self) -> himuon_hparams:
        return himuon_hparams(self.K, self.a, self.b, self.c, self.eps, self.beta, int(self.nesterov),
                              self.lr, self.wd, self.scale_c)


# ----------------------------------------------------------------------------- C-ABI mirrors

def himuon_supported_tile_sizes(dtype_code: int, path: int = HIMUON_PATH_AUTO) -> List[int]:
    mask = _lib().himuon_supported_tile_sizes(dtype_code, path)
    return [16 << i for i in range(16) if mask & (1 << i)]


def himuon_launch_count() -> int:
    return int(_lib().himuon_launch_count())


def himuon_plan_chunks(n_items: int, bytes_per_item: int, fixed_bytes: int, cap_bytes: int) -> List[int]:
    """Chunk offsets [0, ..., n_items] of the memory-bounded chunking rule."""
    lib = _lib()
    n = C.c_int32(0)
    _check(lib.himuon_plan_chunks(n_items, bytes_per_item, fixed_bytes, cap_bytes, C.byref(n), None, 0),
           "himuon_plan_chunks")
    offs = np.zeros(n.value + 1, dtype=np.int64)
    _check(lib.himuon_plan_chunks(n_items, bytes_per_item, fixed_bytes, cap_bytes, C.byref(n),
                                  offs.ctypes.data, n.value + 1), "himuon_plan_chunks")
    return [int(x) for x in offs]


class Plan:
    """Owner of a `himuon_plan*` (himuon_plan_create .. himuon_plan_destroy)."""

    def __init__(self, layers: Sequence[himuon_layer], T_default: int, path: int = HIMUON_PATH_AUTO,
                 workspace_cap_bytes: int = 0):
        lib = self._lib = _lib()      # a plan stays with the library that created it
        arr = (himuon_layer * len(layers))(*layers)
        h = C.c_void_p()
        _check(lib.himuon_plan_create(arr, len(layers), T_default, path, workspace_cap_bytes, C.byref(h)),
               "himuon_plan_create")
        self._h = h
        self._keep = []          # tensors the descriptors point to
        self.workspace = None
        nt, nb, nc, wb = C.c_int64(), C.c_int32(), C.c_int32(), C.c_size_t()
        _check(lib.himuon_plan_info(h, C.byref(nt), C.byref(nb), C.byref(nc), C.byref(wb)), "himuon_plan_info")
        self.n_tiles, self.n_buckets, self.n_chunks, self.workspace_bytes = nt.value, nb.value, nc.value, wb.value

    @classmethod
    def from_tensors(cls, Ws, Gs, Ms, T_default: int, T_per_layer: Optional[Sequence[int]] = None,
                     path: int = HIMUON_PATH_AUTO, workspace_cap_bytes: int = 0,
                     Tw_per_layer: Optional[Sequence[int]] = None) -> "Plan":
        """Tw_per_layer: tile width per layer for rectangular tiles (T rows x T_w columns); 0 / None = square."""
        layers = []
        for i, (w, g) in enumerate(zip(Ws, Gs)):
            m = Ms[i] if Ms is not None else None
            layers.append(himuon_layer(mat_of(w), mat_of(g), mat_of(m), T_per_layer[i] if T_per_layer else 0,
                                       Tw_per_layer[i] if Tw_per_layer else 0))
        p = cls(layers, T_default, path, workspace_cap_bytes)
        p._keep = [Ws, Gs, Ms]
        return p

    def worklist(self) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
        """(lrc [n_tiles,3] int32, chunk_offsets [n_chunks+1] int64, chunk_T [n_chunks] int32)."""
        lrc = np.zeros((self.n_tiles, 3), dtype=np.int32)
        offs = np.zeros(self.n_chunks + 1, dtype=np.int64)
        cT = np.zeros(max(self.n_chunks, 1), dtype=np.int32)
        _check(self._lib.himuon_plan_worklist(self._h, lrc.ctypes.data, offs.ctypes.data, cT.ctypes.data),
               "himuon_plan_worklist")
        return lrc, offs, cT[: self.n_chunks]

    def bind(self, workspace: Optional[torch.Tensor] = None, stream=None) -> "Plan":
        if workspace is None:
            workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device="cuda")
        off = (-workspace.data_ptr()) % 128
        self.workspace = workspace
        _check(self._lib.himuon_plan_bind(self._h, workspace.data_ptr() + off, workspace.numel() - off,
                                       _stream_ptr(stream)), "himuon_plan_bind")
        return self

    def step(self, hp: HParams, stream=None):
        c = hp.to_c()
        _check(self._lib.himuon_step(self._h, C.byref(c), _stream_ptr(stream)), "himuon_step")

    def phi(self, hp: HParams, stream=None):
        c = hp.to_c()
        _check(self._lib.himuon_phi(self._h, C.byref(c), _stream_ptr(stream)), "himuon_phi")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.himuon_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def himuon_ns_tiles(tiles_in: torch.Tensor, tiles_out: Optional[torch.Tensor] = None, K: int = 5,
                    a: float = NS_COEFFS[0], b: float = NS_COEFFS[1], c: float = NS_COEFFS[2],
                    eps: float = 1e-7, path: int = HIMUON_PATH_AUTO, workspace: Optional[torch.Tensor] = None,
                    stream=None) -> torch.Tensor:
    """Packed [N, T, T] tiles -> Phi_K(tiles) (the Fig. 7 workload)."""
    if tiles_in.dim() != 3 or tiles_in.shape[1] != tiles_in.shape[2] or not tiles_in.is_contiguous():
        raise ValueError("tiles_in must be a contiguous [N, T, T] tensor")
    if tiles_out is None:
        tiles_out = torch.empty_like(tiles_in)
    lib = _lib()
    if workspace is None:
        workspace = torch.empty(lib.himuon_ns_tiles_workspace_bytes() + 256, dtype=torch.uint8,
                                device=tiles_in.device)
    off = (-workspace.data_ptr()) % 128
    N, T = tiles_in.shape[0], tiles_in.shape[1]
    _check(lib.himuon_ns_tiles(tiles_in.data_ptr(), tiles_out.data_ptr(), N, T, _dtype_code(tiles_in.dtype),
                               path, K, a, b, c, eps, workspace.data_ptr() + off, workspace.numel() - off,
                               _stream_ptr(stream)), "himuon_ns_tiles")
    # the workspace must outlive the asynchronous launch
    tiles_out._himuon_ws = workspace
    return tiles_out


def himuon_ns_tiles_static(tiles_in: torch.Tensor, tiles_out: torch.Tensor, K: int = 5, a: float = NS_COEFFS[0],
                           b: float = NS_COEFFS[1], c: float = NS_COEFFS[2], eps: float = 1e-7, stream=None) -> torch.Tensor:
    """himuon_ns_tiles without a workspace and without any allocation (here or in the library): bf16 [N, T, T] tiles,
    N <= himuon_ns_tiles_static_max_tiles(T); the scratch is a static device array inside the library (himuon.h)."""
    if tiles_in.dim() != 3 or tiles_in.shape[1] != tiles_in.shape[2] or not tiles_in.is_contiguous():
        raise ValueError("tiles_in must be a contiguous [N, T, T] tensor")
    if tiles_in.dtype != torch.bfloat16 or tiles_out.dtype != torch.bfloat16 or tiles_out.shape != tiles_in.shape or not tiles_out.is_contiguous():
        raise ValueError("tiles_in / tiles_out must be contiguous bf16 tensors of the same shape")
    lib = _lib()
    st = lib.himuon_ns_tiles_static(tiles_in.data_ptr(), tiles_out.data_ptr(), tiles_in.shape[0], tiles_in.shape[1],
                                    K, a, b, c, eps, _stream_ptr(stream))
    if st == HIMUON_ERR_WORKSPACE_TOO_SMALL:          # the library spells out the limit
        err = HimuonError(st, "himuon_ns_tiles_static")
        err.args = (f"{err.args[0]} ({lib.himuon_last_cuda_error().decode()})",)
        raise err
    _check(st, "himuon_ns_tiles_static")
    return tiles_out


def himuon_ns_tiles_static_max_tiles(T: int) -> int:
    return int(_lib().himuon_ns_tiles_static_max_tiles(T))


def debug_set_stage(kernel: str, stage: int):
    """Accumulator-dump stage of the T = 128 kernels (`kernel` = "tc128" | "tc128_fp8"); exists only in the
    -DHIMUON_DEBUG_STAGES library (see `use_library`, `build.build_debug`)."""
    fn = getattr(_lib(), f"himuon_debug_set_{kernel}_stage")
    fn.restype = None
    fn.argtypes = [C.c_int]
    fn(stage)
