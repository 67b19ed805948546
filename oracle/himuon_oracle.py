"""float64 CPU oracle for HiMuon's tiled Newton-Schulz update (arxiv/paper_2606_27216).

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and bench.py's
`cpu_baseline` / `--impl reference` legs may import this file.  The product path
(`paper_2606_27216_b200/`) never imports it and it never imports the product path; the two
share no code (only the seeded input generators in `himuon_inputs.py`, which hold none of the
method's arithmetic).

Plain, slow, obviously-correct numpy in float64.  Each function is the definition in PAPER.md
written out; there is no blocking, batching, fusion or reordering beyond what the cited passage
states.  Where the paper is silent / garbled the reading is the one listed in DESIGN.md
("Readings of the paper", Q1..Q18 from SURVEY.md section 8(c)).

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): SVD closed form, T>=max(H,W) => full map,
transpose equivariance, tile independence, T=1 scalar iterate in exact rational arithmetic,
block-diagonal inputs, zero tiles, ragged == padded, scale invariance / oddness, orthogonal
invariance, semi-orthogonal input, step identities, and the paper's printed planner numbers
(1680 tiles / 5376 tiles -> 2 x 2688 / 196 calls; tests/golden/paper_planner_numbers.txt).
No function in this file is "parity unpinned".
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Optional, Sequence, Tuple

import numpy as np

# PAPER.md:74, Eq. (2.3): (a, b, c) = (3.4445, -4.7750, 2.0315)
NS_A, NS_B, NS_C = 3.4445, -4.7750, 2.0315


# ----------------------------------------------------------------------------- Phi_K

def phi(A: np.ndarray, K: int = 5, a: float = NS_A, b: float = NS_B, c: float = NS_C,
        eps: float = 0.0) -> np.ndarray:
    """K-step quintic Newton-Schulz map Phi_K (section 2.2, Eq. 2.2-2.3).

    X_0 = A / ||A||_F   ("||A||_E" there is a garble of the Frobenius norm, reading Q3;
                         eps is ADDED to the norm, reading Q2; eps = 0 is the paper's definition)
    X_{k+1} = (a I + b X_k X_k^T + c (X_k X_k^T)^2) X_k            (Eq. 2.2)
    If H > W the recurrence is applied to A^T and transposed back.
    Phi_K(0) = 0.
    """
    A = np.asarray(A, dtype=np.float64)
    H, W = A.shape
    nrm = math.sqrt(float(np.sum(A * A)))
    if nrm == 0.0:
        return np.zeros_like(A)
    if H > W:
        return phi(A.T, K, a, b, c, eps).T
    X = A / (nrm + eps)
    I = np.eye(H, dtype=np.float64)
    for _ in range(K):
        G = X @ X.T
        X = (a * I + b * G + c * (G @ G)) @ X
    return X


# ----------------------------------------------------------------------------- B_T and B_T^{-1}

def tile_grid(H: int, W: int, T: int) -> Tuple[int, int]:
    """R = ceil(H/T), C = ceil(W/T)."""
    return -(-H // T), -(-W // T)


def tile(A: np.ndarray, T: int) -> np.ndarray:
    """Tiling operator B_T: zero-pad to (RT)x(CT), cut an R x C grid of TxT tiles.

    Returns an array of shape [R, C, T, T]; tile (r, c) holds padded rows rT..rT+T-1 and
    columns cT..cT+T-1 (0-based r, c; the paper writes r = 1..R, c = 1..C, reading Q4).
    """
    A = np.asarray(A, dtype=np.float64)
    H, W = A.shape
    R, C = tile_grid(H, W, T)
    P = np.zeros((R * T, C * T), dtype=np.float64)
    P[:H, :W] = A
    out = np.empty((R, C, T, T), dtype=np.float64)
    for r in range(R):
        for c in range(C):
            out[r, c] = P[r * T:(r + 1) * T, c * T:(c + 1) * T]
    return out


def untile(tiles: np.ndarray, H: int, W: int) -> np.ndarray:
    """Inverse operator B_T^{-1}: reassemble the tiles, then remove the padding."""
    R, C, T, T2 = tiles.shape
    assert T == T2
    P = np.empty((R * T, C * T), dtype=np.float64)
    for r in range(R):
        for c in range(C):
            P[r * T:(r + 1) * T, c * T:(c + 1) * T] = tiles[r, c]
    return P[:H, :W].copy()


def is_full_branch(H: int, W: int, T: Optional[int]) -> bool:
    """T = infinity (None) or T >= max(H, W) selects the full-matrix branch (Alg. 4.1 l.10)."""
    return T is None or T >= max(H, W)


def phi_tiled(A: np.ndarray, T: Optional[int], K: int = 5, a: float = NS_A, b: float = NS_B,
              c: float = NS_C, eps: float = 0.0) -> np.ndarray:
    """Tiled map Phi_{K,T} (Eq. 4.1-4.3).

    Finite T < max(H,W): Phi_{K,T}(A) = B_T^{-1}({Phi_K(A_rc)}), implemented literally with
    zero padding.  T = infinity or T >= max(H,W): the full-matrix branch Phi_K(A) (Eq. 4.3 and
    PAPER.md:243, "this case is therefore identified with the full-matrix branch").
    """
    A = np.asarray(A, dtype=np.float64)
    H, W = A.shape
    if is_full_branch(H, W, T):
        return phi(A, K, a, b, c, eps)
    tiles = tile(A, T)
    R, C = tiles.shape[:2]
    out = np.empty_like(tiles)
    for r in range(R):
        for cc in range(C):
            out[r, cc] = phi(tiles[r, cc], K, a, b, c, eps)
    return untile(out, H, W)


def phi_tiles(tiles: np.ndarray, K: int = 5, a: float = NS_A, b: float = NS_B, c: float = NS_C,
              eps: float = 0.0) -> np.ndarray:
    """Phi_K applied independently to each tile of a packed [N, T, T] batch ("tilewise NS", Alg. 4.1 l.15)."""
    tiles = np.asarray(tiles, dtype=np.float64)
    out = np.empty_like(tiles)
    for n in range(tiles.shape[0]):
        out[n] = phi(tiles[n], K, a, b, c, eps)
    return out


# ----------------------------------------------------------------------------- Algorithm 4.1

@dataclass
class HParams:
    """Hyper-parameters of Algorithm 4.1 with the paper's defaults."""
    lr: float = 0.02          # eta
    beta: float = 0.95        # momentum
    nesterov: bool = True
    wd: float = 0.0           # lambda (decoupled weight decay)
    K: int = 5
    a: float = NS_A
    b: float = NS_B
    c: float = NS_C           # NS coefficient c (reading Q6: not the scaling constant)
    eps: float = 0.0
    scale_c: float = 0.2      # scaling constant "c" of section 4.2


def tau(H: int, W: int, T: Optional[int], scale_c: float = 0.2) -> float:
    """Update scaling tau_l(T) (section 4.2):
    c*sqrt(max(H,W)) if T >= max(H,W) (or T = infinity), else c*sqrt(T).  One scalar per matrix,
    shared by all tiles including edge tiles (reading Q8)."""
    if is_full_branch(H, W, T):
        return scale_c * math.sqrt(max(H, W))
    return scale_c * math.sqrt(T)


def momentum(G: np.ndarray, M_prev: np.ndarray, beta: float, nesterov: bool):
    """M_t = beta M_{t-1} + G_t; Ghat = G_t + beta M_t if Nesterov else M_t
    (Alg. 4.1 l.4-9; undamped form and NEW M_t in the look-ahead, reading Q10)."""
    G = np.asarray(G, dtype=np.float64)
    M = beta * np.asarray(M_prev, dtype=np.float64) + G
    Ghat = G + beta * M if nesterov else M
    return M, Ghat


def step(W: np.ndarray, G: np.ndarray, M_prev: np.ndarray, hp: HParams, T: Optional[int]):
    """One HiMuon update of one matrix parameter (Algorithm 4.1 l.4-20, Eq. 4.6).

    Returns (W_t, M_t, U_t) with U_t = Phi_{K,T}(Ghat_t) and
    W_t = (1 - eta*lambda) W_{t-1} - eta * tau * U_t  (both terms see W_{t-1}, reading Q9).
    No intermediate rounding (reading Q11): inputs are whatever float64 values the caller decoded.
    """
    W = np.asarray(W, dtype=np.float64)
    H, Wd = W.shape
    M, Ghat = momentum(G, M_prev, hp.beta, hp.nesterov)
    U = phi_tiled(Ghat, T, hp.K, hp.a, hp.b, hp.c, hp.eps)
    t = tau(H, Wd, T, hp.scale_c)
    W_new = (1.0 - hp.lr * hp.wd) * W - hp.lr * t * U
    return W_new, M, U


# ----------------------------------------------------------------------------- rectangular tiles (T_h, T_w)

def phi_tiled_rect(A: np.ndarray, Th: int, Tw: int, K: int = 5, a: float = NS_A, b: float = NS_B,
                   c: float = NS_C, eps: float = 0.0) -> np.ndarray:
    """Tiled map with rectangular tiles (T_h, T_w) ("Rectangular tiles (T_h, T_w) are used only in the
    tile-shape study of Figure 8; elsewhere T_h = T_w = T").

    The same construction as B_T with the two tile extents decoupled: zero-pad to (R T_h) x (C T_w),
    R = ceil(H / T_h), C = ceil(W / T_w), apply Phi_K to every T_h x T_w tile (Phi_K transposes a tall tile
    internally), reassemble, remove the padding.  T_h >= H and T_w >= W is one tile = the whole
    matrix, i.e. the full-matrix branch."""
    A = np.asarray(A, dtype=np.float64)
    H, W = A.shape
    R, C = -(-H // Th), -(-W // Tw)
    P = np.zeros((R * Th, C * Tw), dtype=np.float64)
    P[:H, :W] = A
    Q = np.empty_like(P)
    for r in range(R):
        for cc in range(C):
            Q[r * Th:(r + 1) * Th, cc * Tw:(cc + 1) * Tw] = phi(P[r * Th:(r + 1) * Th, cc * Tw:(cc + 1) * Tw], K, a, b, c, eps)
    return Q[:H, :W].copy()


def tau_rect(H: int, W: int, Th: int, Tw: int, scale_c: float = 0.2) -> float:
    """tau = c sqrt(max(T_h, T_w)) for rectangular tiles; c sqrt(max(H, W)) when one tile covers
    the matrix (full-matrix branch)."""
    if Th >= H and Tw >= W:
        return scale_c * math.sqrt(max(H, W))
    return scale_c * math.sqrt(max(Th, Tw))


def step_rect(W: np.ndarray, G: np.ndarray, M_prev: np.ndarray, hp: "HParams", Th: int, Tw: int):
    """Algorithm 4.1 with rectangular tiles: momentum, Phi over (T_h, T_w) tiles, update
    W' = (1 - lr wd) W - lr tau U (Eq. 4.6) with tau_rect.  Returns (W', M', U)."""
    M_new, G_hat = momentum(G, M_prev, hp.beta, hp.nesterov)
    U = phi_tiled_rect(G_hat, Th, Tw, hp.K, hp.a, hp.b, hp.c, hp.eps)
    t = tau_rect(G.shape[0], G.shape[1], Th, Tw, hp.scale_c)
    W_new = (1.0 - hp.lr * hp.wd) * np.asarray(W, dtype=np.float64) - hp.lr * t * U
    return W_new, M_new, U


# ----------------------------------------------------------------------------- execution plan (host logic)

def enumerate_tiles(shapes: Sequence[Tuple[int, int]], T_per_layer: Sequence[Optional[int]]) -> List[Tuple[int, int, int]]:
    """Cross-layer work list (section 4.4.2): every layer's tiles flattened, in
    the layer order of the descriptor table, then r-major (index = r*C + c).  A full-branch layer
    (T >= max(H,W)) contributes a single entry (l, 0, 0) (R = C = 1)."""
    out = []
    for l, ((H, W), T) in enumerate(zip(shapes, T_per_layer)):
        if is_full_branch(H, W, T):
            out.append((l, 0, 0))
            continue
        R, C = tile_grid(H, W, T)
        for r in range(R):
            for c in range(C):
                out.append((l, r, c))
    return out


def chunk_offsets(n_items: int, bytes_per_item: int, cap_bytes: int, fixed_bytes: int = 0) -> List[int]:
    """Memory-bounded chunking: split n_items into the FEWEST chunks whose
    workspace (fixed_bytes + items * bytes_per_item) fits cap_bytes; chunks are balanced, as the
    paper's worked example shows (5376 tiles -> two chunks of 2688, not a greedy fill; reading
    Q14).  Returns offsets [0, ..., n_items] (len = n_chunks + 1).  Raises if one item cannot fit.
    """
    if n_items == 0:
        return [0]
    room = cap_bytes - fixed_bytes
    if bytes_per_item <= 0:
        per_chunk_max = n_items
    else:
        per_chunk_max = room // bytes_per_item
    if per_chunk_max < 1:
        raise ValueError("workspace cap too small for a single tile")
    n_chunks = -(-n_items // per_chunk_max)
    base, rem = divmod(n_items, n_chunks)
    offs = [0]
    for i in range(n_chunks):
        offs.append(offs[-1] + base + (1 if i < rem else 0))
    return offs


def per_tile_rel_fro_error(U_test: np.ndarray, U_ref: np.ndarray, T: int) -> np.ndarray:
    """Per-tile relative Frobenius error ||U_test_rc - U_ref_rc||_F / ||U_ref_rc||_F on the B_T grid
    (the parity metric of BASELINE.json north_star).  Tiles whose reference is exactly zero report
    the absolute error.  Returns an [R, C] array."""
    H, W = U_ref.shape
    if is_full_branch(H, W, T):
        T = max(H, W)
    d = tile(np.asarray(U_test, dtype=np.float64) - U_ref, T)
    r = tile(U_ref, T)
    num = np.sqrt(np.sum(d * d, axis=(2, 3)))
    den = np.sqrt(np.sum(r * r, axis=(2, 3)))
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), num)
