"""Process pool over the float64 oracle for the full-size parity tests (test infrastructure; SURVEY.md 8(d):
"stream layer by layer with a process pool across all cores").

The oracle is called as it stands (one `O.step` per tile); the pool only spreads tiles over the host cores.
This module imports numpy and `oracle/` only - no torch - so that `spawn`ed workers start fast and never
touch CUDA.  Tiles travel as raw bf16 bit patterns (uint16) and are decoded exactly to float64 in the worker.
"""
from __future__ import annotations

import multiprocessing as mp
import os
from concurrent.futures import ProcessPoolExecutor
from typing import Dict, List, Sequence, Tuple

import numpy as np

from oracle import himuon_oracle as O

BF16_ULP = 2.0 ** -8


def bf16_bits_to_f64(u: np.ndarray) -> np.ndarray:
    """uint16 bf16 bit patterns -> float64, exactly."""
    return (u.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def _pad(x: np.ndarray, T: int) -> np.ndarray:
    out = np.zeros((T, T), dtype=np.float64)     # B_T zero padding
    out[: x.shape[0], : x.shape[1]] = x
    return out


def _check_batch(job) -> List[Tuple[float, float, bool]]:
    """One batch of tiles of a W0 = 0 step.  Per tile: (relative Frobenius error of the recovered U against the
    oracle's U, worst |M'_gpu - M'_ref| / allowance, all outputs finite)."""
    hpd, T, tau, tiles = job
    ohp = O.HParams(**hpd)
    out = []
    for (g, m0, w1, m1) in tiles:
        G, M0 = _pad(bf16_bits_to_f64(g), T), _pad(bf16_bits_to_f64(m0), T)
        W1, M1 = _pad(bf16_bits_to_f64(w1), T), _pad(bf16_bits_to_f64(m1), T)
        # a T x T block at tile size T is exactly one tile (R = C = 1, same tau = c_s sqrt(T), Eq. 4.6)
        Wr, Mr, Ur = O.step(np.zeros((T, T)), G, M0, ohp, T)
        U_gpu = -W1 / (ohp.lr * tau)                       # W0 = 0  =>  W' = -lr tau U, one RNE rounding
        nu = np.linalg.norm(Ur)
        err_u = float(np.linalg.norm(U_gpu - Ur) / nu) if nu > 0 else float(np.abs(U_gpu).max())
        m_tol = BF16_ULP * np.abs(Mr) + 2.0 ** -21 * (np.abs(ohp.beta * M0) + np.abs(G)) + 1e-30   # reading Q11
        m_ratio = float(np.max(np.abs(M1 - Mr) / m_tol))
        out.append((err_u, m_ratio, bool(np.all(np.isfinite(W1)) and np.all(np.isfinite(M1)))))
    return out


def check_tiles_w0(hp: Dict, T: int, tau: float, tiles: Sequence[Tuple[np.ndarray, np.ndarray, np.ndarray, np.ndarray]],
                   batch: int = 32, workers: int | None = None) -> np.ndarray:
    """Run `_check_batch` over all tiles on a pool of single-threaded workers; returns an [n, 3] array."""
    workers = workers or len(os.sched_getaffinity(0))
    jobs = [(hp, T, tau, tiles[i:i + batch]) for i in range(0, len(tiles), batch)]
    saved = {k: os.environ.get(k) for k in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS")}
    for k in saved:
        os.environ[k] = "1"                                # one BLAS thread per worker: the pool is the parallelism
    try:
        with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as pool:
            res = [r for part in pool.map(_check_batch, jobs) for r in part]
    finally:
        for k, v in saved.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v
    return np.array([(a, b, float(c)) for a, b, c in res], dtype=np.float64).reshape(-1, 3)
