"""Seeded synthetic inputs for the HiMuon hot path (shared by oracle tests, GPU tests and bench.py).

This module holds NONE of the method's arithmetic (no Newton-Schulz, no tiling, no momentum,
no update rule).  It only draws random matrices with the shapes / value distributions named in
BASELINE.json `configs` and SURVEY.md section 8(d), and converts between storage dtypes.

The paper's own workloads are bf16 Gaussian matrices / tiles for the kernel studies
(section 6.3) and fresh random Gaussian gradients for the optimizer-step study
(section 6.4).  Its training data and models (FineWeb, Qwen3) are not available and
not needed: the recipes below stand in for them.

Every tensor is drawn from its own torch.Generator seeded with
    seed_cfg * 1_000_003 + layer_index * 16 + tensor_id
(tensor_id: 0 = G, 1 = M_prev, 2 = W, 3 = left factor, 4 = right factor, 5 = row scales).
CPU and CUDA generators produce different streams; parity never relies on them agreeing: inputs
are generated once on one device and the SAME BITS are copied to the other side.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np
import torch

TENSOR_G, TENSOR_M, TENSOR_W, TENSOR_U, TENSOR_V, TENSOR_S = 0, 1, 2, 3, 4, 5


def _gen(device, seed_cfg: int, layer_index: int, tensor_id: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed_cfg * 1_000_003 + layer_index * 16 + tensor_id)
    return g


def _randn(shape, device, gen) -> torch.Tensor:
    return torch.randn(shape, device=device, dtype=torch.float32, generator=gen)


# ----------------------------------------------------------------------------- dtype helpers

def to_f64_numpy(t: torch.Tensor) -> np.ndarray:
    """Exact decode of a stored tensor (bf16 / fp32) to a float64 numpy array."""
    return t.detach().to("cpu").to(torch.float64).numpy()


def bf16_round_f64(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even a float array to bf16 and return the float64 values (storage model)."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).to(torch.float32)
    return t.to(torch.bfloat16).to(torch.float64).numpy()


# ----------------------------------------------------------------------------- matrix recipes

def gaussian(H: int, W: int, *, seed_cfg: int, layer_index: int = 0, tensor_id: int = TENSOR_G,
             dtype=torch.float32, device="cpu", scale: float = 1.0) -> torch.Tensor:
    """i.i.d. N(0, scale^2) entries (config 1: fp32 256x512 from seed 0)."""
    x = _randn((H, W), device, _gen(device, seed_cfg, layer_index, tensor_id))
    if scale != 1.0:
        x = x * scale
    return x.to(dtype)


def lowrank_plus_noise(H: int, W: int, rank: int, *, seed_cfg: int, layer_index: int,
                       tensor_id: int, noise: float = 0.1, dtype=torch.bfloat16,
                       device="cpu") -> torch.Tensor:
    """U V^T / sqrt(rank) + noise * N(0,1); U in R^{H x rank}, V in R^{W x rank} i.i.d. N(0,1).

    Configs 2/4/5 ("rank-16 Gaussian factors (unit variance, scaled 1/sqrt(16)) plus 0.1*N(0,1)").
    The factor / noise sub-streams are derived from tensor_id so that G and M_prev differ.
    """
    gu = _gen(device, seed_cfg, layer_index, TENSOR_U + 8 * tensor_id)
    gv = _gen(device, seed_cfg, layer_index, TENSOR_V + 8 * tensor_id)
    gn = _gen(device, seed_cfg, layer_index, tensor_id)
    U = _randn((H, rank), device, gu)
    V = _randn((W, rank), device, gv)
    x = (U @ V.t()) * (1.0 / math.sqrt(rank))
    del U, V
    x.add_(_randn((H, W), device, gn), alpha=noise)
    return x.to(dtype)


def row_scaled_gaussian(H: int, W: int, *, seed_cfg: int, layer_index: int = 0,
                        sigma_log: float = 0.5, dtype=torch.bfloat16, device="cpu") -> torch.Tensor:
    """N(0,1) * sigma_row with sigma_row ~ LogNormal(0, sigma_log) per row (config 3)."""
    gs = _gen(device, seed_cfg, layer_index, TENSOR_S)
    gn = _gen(device, seed_cfg, layer_index, TENSOR_G)
    s = torch.exp(sigma_log * _randn((H, 1), device, gs))
    x = _randn((H, W), device, gn) * s
    return x.to(dtype)


def integer_tags(H: int, W: int, *, layer_index: int = 0, dtype=torch.bfloat16,
                 device="cpu") -> torch.Tensor:
    """Integer-tagged matrix for bit-exact indexing tests: tag = f(layer,i,j) mod 251, +1.

    Values are integers in [1, 251], exactly representable in bf16 (8 significant bits cover
    integers up to 256) and in fp32.
    """
    i = torch.arange(H, device=device, dtype=torch.int64).unsqueeze(1)
    j = torch.arange(W, device=device, dtype=torch.int64).unsqueeze(0)
    tag = (i * 131 + j * 7 + layer_index * 53) % 251 + 1
    return tag.to(torch.float32).to(dtype)


# ----------------------------------------------------------------------------- parameter sets

@dataclass
class LayerSpec:
    name: str
    H: int
    W: int
    T: int = 0          # 0 = plan-wide default


@dataclass
class ParamSetSpec:
    name: str
    seed_cfg: int
    rank: int
    layers: List[LayerSpec] = field(default_factory=list)

    @property
    def n_elements(self) -> int:
        return sum(l.H * l.W for l in self.layers)


def gpt2_small_spec() -> ParamSetSpec:
    """Config 2: 12 layers x {Wq,Wk,Wv,Wo 768x768, W_fc 768x3072, W_proj 3072x768}, rank 16, seed 1."""
    L = []
    for b in range(12):
        for n in ("q", "k", "v", "o"):
            L.append(LayerSpec(f"h{b}.{n}", 768, 768))
        L.append(LayerSpec(f"h{b}.fc", 768, 3072))
        L.append(LayerSpec(f"h{b}.proj", 3072, 768))
    return ParamSetSpec("gpt2-small", 1, 16, L)


def gpt2_xl_spec(n_blocks: int = 48) -> ParamSetSpec:
    """Config 4: 48 layers x {4x 1600x1600, 1600x6400, 6400x1600}, rank 32, seed 3 (ragged at T=128)."""
    L = []
    for b in range(n_blocks):
        for n in ("q", "k", "v", "o"):
            L.append(LayerSpec(f"h{b}.{n}", 1600, 1600))
        L.append(LayerSpec(f"h{b}.fc", 1600, 6400))
        L.append(LayerSpec(f"h{b}.proj", 6400, 1600))
    return ParamSetSpec("gpt2-xl", 3, 32, L)


def llama3_8b_spec(n_blocks: int = 32, schedule: bool = False) -> ParamSetSpec:
    """Config 5: 32 layers x {q,o 4096^2; k,v 1024x4096; gate,up 14336x4096; down 4096x14336}.

    rank 64, seed 4.  schedule=True attaches the per-layer-type tile sizes of DESIGN.md reading
    Q13 (k,v -> 64; q,o -> 128; gate,up,down -> 256); otherwise T=0 (plan-wide default).
    """
    tq, tkv, tmlp = (128, 64, 256) if schedule else (0, 0, 0)
    L = []
    for b in range(n_blocks):
        L.append(LayerSpec(f"l{b}.q", 4096, 4096, tq))
        L.append(LayerSpec(f"l{b}.k", 1024, 4096, tkv))
        L.append(LayerSpec(f"l{b}.v", 1024, 4096, tkv))
        L.append(LayerSpec(f"l{b}.o", 4096, 4096, tq))
        L.append(LayerSpec(f"l{b}.gate", 14336, 4096, tmlp))
        L.append(LayerSpec(f"l{b}.up", 14336, 4096, tmlp))
        L.append(LayerSpec(f"l{b}.down", 4096, 14336, tmlp))
    return ParamSetSpec("llama3-8b", 4, 64, L)


def qwen3_block_shapes() -> dict:
    """PAPER.md:361-368, Table 2 (output x input) -- used only by the planner's worked example."""
    return {
        "0.6B": [(2048, 1024), (1024, 1024), (1024, 1024), (1024, 2048),
                 (3072, 1024), (3072, 1024), (1024, 3072)],
        "1.7B": [(2048, 2048), (1024, 2048), (1024, 2048), (2048, 2048),
                 (6144, 2048), (6144, 2048), (2048, 6144)],
        "4B": [(4096, 2560), (1024, 2560), (1024, 2560), (2560, 4096),
               (9728, 2560), (9728, 2560), (2560, 9728)],
    }


def make_layer_tensors(spec: ParamSetSpec, layer_index: int, *, dtype=torch.bfloat16,
                       device="cpu") -> Tuple[torch.Tensor, torch.Tensor, torch.Tensor]:
    """(W, G, M_prev) for one layer of a parameter set (reading Q17)."""
    l = spec.layers[layer_index]
    G = lowrank_plus_noise(l.H, l.W, spec.rank, seed_cfg=spec.seed_cfg, layer_index=layer_index,
                           tensor_id=TENSOR_G, dtype=dtype, device=device)
    M = lowrank_plus_noise(l.H, l.W, spec.rank, seed_cfg=spec.seed_cfg, layer_index=layer_index,
                           tensor_id=TENSOR_M, dtype=dtype, device=device)
    W = gaussian(l.H, l.W, seed_cfg=spec.seed_cfg, layer_index=layer_index, tensor_id=TENSOR_W,
                 dtype=dtype, device=device, scale=0.02)
    return W, G, M


def make_param_set(spec: ParamSetSpec, *, dtype=torch.bfloat16, device="cpu",
                   layers: Sequence[int] | None = None):
    """Lists (W, G, M_prev) for the selected layers (default: all)."""
    idx = range(len(spec.layers)) if layers is None else layers
    Ws, Gs, Ms = [], [], []
    for i in idx:
        W, G, M = make_layer_tensors(spec, i, dtype=dtype, device=device)
        Ws.append(W); Gs.append(G); Ms.append(M)
    return Ws, Gs, Ms


# ----------------------------------------------------------------------------- capacity diagnostic workload
# The one-step linear associative-memory benchmark the paper uses as its capacity diagnostic
# (section 5.1; instance sizes PAPER.md:410 section 6.5).  This is the WORKLOAD around
# the map - key/value embeddings, the minibatch, the gradient of the cross-entropy loss at W_0 = 0 and the
# recovered-item count - and holds none of the method's arithmetic: the update map is applied by the
# caller (the oracle in the CPU pins, the CUDA path in the GPU tests).

@dataclass
class AssocMemoryProblem:
    U: np.ndarray          # [N, d] values u_j  ~ N(0, I/d)
    V: np.ndarray          # [N, d] keys   v_i  ~ N(0, I/d)
    idx: np.ndarray        # [B] sampled item indices, p_i ~ i^-alpha (with replacement)
    G0: np.ndarray         # [d, d] minibatch gradient of the cross-entropy loss at W_0 = 0, float64


def assoc_memory_problem(d: int, N: int, alpha: float, B: int, seed: int) -> AssocMemoryProblem:
    """Logits of key v_i are u_j^T W v_i; at W_0 = 0 the softmax is uniform, so the
    gradient of the mean cross-entropy over the minibatch is
        G_0 = (1/B) sum_b (ubar - u_{i_b}) v_{i_b}^T,   ubar = (1/N) sum_j u_j,
    built in float64 ("constructed in fp64 and held fixed across precision variants")."""
    g = np.random.default_rng(1_000_003 * 7 + seed)
    V = g.standard_normal((N, d)) / math.sqrt(d)
    U = g.standard_normal((N, d)) / math.sqrt(d)
    p = np.arange(1, N + 1, dtype=np.float64) ** (-alpha)
    p /= p.sum()
    idx = g.choice(N, size=B, p=p)
    cnt = np.bincount(idx, minlength=N).astype(np.float64)
    ubar = U.mean(axis=0)
    G0 = ((cnt[:, None] * (ubar[None, :] - U)).T @ V) / B
    return AssocMemoryProblem(U=U, V=V, idx=idx, G0=G0)


def recovered_items(prob: AssocMemoryProblem, W1: np.ndarray) -> int:
    """Number of items k with argmax_j u_j^T W_1 v_k = k."""
    logits = (prob.U @ W1) @ prob.V.T          # [j, k]
    return int((np.argmax(logits, axis=0) == np.arange(prob.U.shape[0])).sum())
