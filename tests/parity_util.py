"""Helpers for the GPU parity tests: run the float64 oracle on the same bits the GPU saw and
compare per tile.  (Test infrastructure; the only place besides bench.py / smoke() that touches oracle/.)"""
from __future__ import annotations

import math
from typing import Optional, Sequence

import numpy as np
import torch

import himuon_inputs as I
from oracle import himuon_oracle as O

TOL_TC = 3e-2      # bf16 tensor-core path, per-tile relative Frobenius error (BASELINE.json north_star)
TOL_FP32 = 1e-4    # fp32 path
BF16_ULP = 2.0 ** -8


def f64(t: torch.Tensor) -> np.ndarray:
    return I.to_f64_numpy(t)


def oracle_hp(hp) -> O.HParams:
    return O.HParams(lr=hp.lr, beta=hp.beta, nesterov=bool(hp.nesterov), wd=hp.wd, K=hp.K, a=float(np.float32(hp.a)),
                     b=float(np.float32(hp.b)), c=float(np.float32(hp.c)), eps=float(np.float32(hp.eps)),
                     scale_c=hp.scale_c)


def tile_err(U_gpu: np.ndarray, U_ref: np.ndarray, T: int) -> np.ndarray:
    return O.per_tile_rel_fro_error(U_gpu, U_ref, T)


def tile_fro(A: np.ndarray, T: int) -> np.ndarray:
    H, W = A.shape
    if O.is_full_branch(H, W, T):
        T = max(H, W)
    t = O.tile(A, T)
    return np.sqrt(np.sum(t * t, axis=(2, 3)))


def check_phi(U_gpu: torch.Tensor, G: torch.Tensor, T: int, hp, tol: float, out_is_bf16: bool):
    """Phi_{K,T}(G) from the GPU against the oracle; returns the max per-tile error."""
    ohp = oracle_hp(hp)
    ref = O.phi_tiled(f64(G), T, ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
    err = tile_err(f64(U_gpu), ref, T)
    assert np.all(np.isfinite(f64(U_gpu))), "non-finite output"
    assert err.max() <= tol, f"per-tile rel Fro error {err.max():.3e} > {tol:.1e} (median {np.median(err):.3e})"
    return float(err.max())


def check_step(W0, G, M0, W1, M1, T: int, hp, tol: float, storage_bf16: bool):
    """One Algorithm-4.1 step (W0,G,M0) -> (W1,M1) from the GPU against the oracle (reading Q11)."""
    ohp = oracle_hp(hp)
    Wr, Mr, Ur = O.step(f64(W0), f64(G), f64(M0), ohp, T)
    m_gpu, w_gpu = f64(M1), f64(W1)
    assert np.all(np.isfinite(m_gpu)) and np.all(np.isfinite(w_gpu))
    # momentum: one rounding on store
    # (relative to the result) plus fp32 arithmetic on the operands (which may cancel)
    m_tol = (BF16_ULP if storage_bf16 else 2.0 ** -22) * np.abs(Mr) + 2.0 ** -21 * (np.abs(ohp.beta * f64(M0)) + np.abs(f64(G))) + 1e-30
    assert np.all(np.abs(m_gpu - Mr) <= m_tol), f"M' off by {np.max(np.abs(m_gpu - Mr) / (np.abs(Mr) + 1e-30)):.3e} rel"
    # weights: per tile,  ||W'_gpu - W'_ref||_F <= round(W'_ref) + lr*tau*tol*||U_ref||_F.  The rounding term is the
    # RMS of one RNE rounding, not a full ulp per element: an element with spacing s (s <= 2^-7 |w| in bf16) is off by
    # a uniform error in [-s/2, s/2], i.e. s/sqrt(12) rms, so ||err||_F <= 2^-7/sqrt(12) ||W'||_F in expectation; the
    # factor (1.1 + 4/sqrt(n)) covers the fluctuation over the n stored elements of the tile (1.1 for a full tile, more
    # for a small ragged block), capped at the hard bound of half a spacing per element (2^-8 ||W'||_F).
    H, Wd = Wr.shape
    tau = O.tau(H, Wd, T, ohp.scale_c)
    dW = tile_fro(w_gpu - Wr, T)
    n_live = np.maximum(tile_fro((Wr != 0).astype(np.float64), T) ** 2, 1.0)
    if storage_bf16:
        rnd = np.minimum((2.0 ** -7 / math.sqrt(12.0)) * (1.1 + 4.0 / np.sqrt(n_live)), BF16_ULP) * tile_fro(Wr, T)
    else:
        rnd = 2.0 ** -22 * tile_fro(Wr, T)
    bound = rnd + abs(ohp.lr) * tau * tol * tile_fro(Ur, T) + 1e-30
    assert np.all(dW <= bound), f"W' tile error ratio {np.max(dW / bound):.3f} > 1"
    return float(np.max(dW / bound))
