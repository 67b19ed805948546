"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (one plan over the
whole parameter set, the config's workspace cap): seeded inputs drawn on the GPU with the config's recipe,
one himuon_step / himuon_phi, then a seeded SAMPLE of tiles (plus every kind of edge tile) is copied back
- inputs before, outputs after - and each sampled tile is checked against the float64 oracle.  Tiles are
independent, so a T x T block cut at a tile boundary with tile size T is exactly
one tile of the full problem (same tau = c_s sqrt(T), Eq. 4.6)."""
import numpy as np
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm
import parity_util as PU

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _need_gpu(min_gb=0):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    if min_gb and torch.cuda.get_device_properties(0).total_memory < min_gb * 2**30:
        pytest.skip(f"needs {min_gb} GB of device memory")


def _sample_tiles(spec, Tl, n, seed):
    """(layer, r, c) picks: n random tiles plus, per distinct layer shape, the last-row / last-column / corner tile."""
    rng = np.random.default_rng(seed)
    picks, seen = set(), set()
    for li, l in enumerate(spec.layers):
        T = Tl[li]
        R, C = -(-l.H // T), -(-l.W // T)
        if (l.H, l.W, T) not in seen:
            seen.add((l.H, l.W, T))
            picks.update({(li, R - 1, C - 1), (li, R - 1, 0), (li, 0, C - 1), (li, 0, 0)})
    while len(picks) < n + 4 * len(seen):
        li = int(rng.integers(len(spec.layers)))
        T = Tl[li]
        l = spec.layers[li]
        picks.add((li, int(rng.integers(-(-l.H // T))), int(rng.integers(-(-l.W // T)))))
    return sorted(picks)


def _cut(t, T, r, c):
    return t[r * T:(r + 1) * T, c * T:(c + 1) * T].clone()


def _run_config_step(spec, T_default, cap_mb, n_sample, seed, path=hm.HIMUON_PATH_AUTO, tol=PU.TOL_TC):
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    Tl = [l.T or T_default for l in spec.layers]
    Ws, Gs, Ms = [], [], []
    for i in range(len(spec.layers)):
        W, G, M = I.make_layer_tensors(spec, i, dtype=torch.bfloat16, device=DEV)
        Ws.append(W); Gs.append(G); Ms.append(M)
    picks = _sample_tiles(spec, Tl, n_sample, seed)
    before = [(_cut(Ws[li], Tl[li], r, c).cpu(), _cut(Gs[li], Tl[li], r, c).cpu(), _cut(Ms[li], Tl[li], r, c).cpu())
              for (li, r, c) in picks]
    plan = hm.Plan.from_tensors(Ws, Gs, Ms, T_default, T_per_layer=Tl if any(l.T for l in spec.layers) else None,
                                path=path, workspace_cap_bytes=cap_mb << 20).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    worst = 0.0
    for (li, r, c), (W0, G0, M0) in zip(picks, before):
        T = Tl[li]
        W1, M1, G1 = _cut(Ws[li], T, r, c).cpu(), _cut(Ms[li], T, r, c).cpu(), _cut(Gs[li], T, r, c).cpu()
        assert torch.equal(G1, G0), "G was modified"
        # a ragged edge block is smaller than T x T: pad it to the tile (B_T zero padding)
        def pad(x):
            out = torch.zeros(T, T, dtype=x.dtype)
            out[:x.shape[0], :x.shape[1]] = x
            return out
        ratio = PU.check_step(pad(W0), pad(G0), pad(M0), pad(W1), pad(M1), T, hp, tol, storage_bf16=True)
        worst = max(worst, ratio)
    return plan, worst, len(picks)


def test_config2_gpt2_small_full_step():
    """BASELINE configs[1]: 72 matrices, 5184 tiles, one cross-layer launch."""
    _need_gpu()
    plan, worst, n = _run_config_step(I.gpt2_small_spec(), 128, 2048, 96, 2)
    assert plan.n_tiles == 5184 and plan.n_chunks == 1 and plan.n_buckets == 1


def test_config4_gpt2_xl_ragged_capped():
    """BASELINE configs[3]: 1600 leaves 64-wide edge tiles at T = 128; 256 MB workspace cap."""
    _need_gpu(40)
    plan, worst, n = _run_config_step(I.gpt2_xl_spec(), 128, 256, 96, 4)
    assert plan.n_tiles == 94848
    assert plan.workspace_bytes <= 256 << 20


@pytest.mark.parametrize("T", [128, 64, 256, 32, 16])
def test_config5_llama3_8b_step(T):
    """BASELINE configs[4] at full size (425 984 tiles at T = 128), 2 GB workspace cap: bench.py's launch."""
    _need_gpu(120)
    plan, worst, n = _run_config_step(I.llama3_8b_spec(), T, 2048, 128, 5)
    assert plan.n_tiles == {128: 425984, 64: 1703936, 256: 106496, 32: 6815744, 16: 27262976}[T]
    assert plan.workspace_bytes <= 2048 << 20


@pytest.mark.parametrize("T", [128, 256])
def test_config5_llama3_8b_step_fp8(T):
    """The same full-size launch on the opt-in e4m3-operand path (HIMUON_PATH_FP8), at its own tolerance (0.15)."""
    _need_gpu(120)
    plan, worst, n = _run_config_step(I.llama3_8b_spec(), T, 2048, 128, 5, path=hm.HIMUON_PATH_FP8, tol=0.15)
    assert plan.n_tiles == {128: 425984, 256: 106496}[T]


@pytest.mark.parametrize("T", [128, 256])
def test_config4_gpt2_xl_ragged_fp8_deterministic(T):
    """GPT-2-XL shapes (64-wide edge tiles) on the e4m3-operand path: two steps from the same bits twice give bitwise
    identical W' and M' (no race between the slots, the prefetches and the stores)."""
    _need_gpu(40)
    spec = I.gpt2_xl_spec(n_blocks=4)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    outs = []
    for rep in range(2):
        Ws, Gs, Ms = [], [], []
        for i in range(len(spec.layers)):
            W, G, M = I.make_layer_tensors(spec, i, dtype=torch.bfloat16, device=DEV)
            Ws.append(W); Gs.append(G); Ms.append(M)
        plan = hm.Plan.from_tensors(Ws, Gs, Ms, T, path=hm.HIMUON_PATH_FP8).bind()
        plan.step(hp)
        plan.step(hp)
        torch.cuda.synchronize()
        outs.append((Ws, Ms))
        plan.destroy()
    for a, b in zip(outs[0][0] + outs[0][1], outs[1][0] + outs[1][1]):
        assert torch.equal(a, b)
        assert bool(torch.isfinite(a.float()).all())


def test_config5_schedule_per_layer_type():
    """Runtime tile schedule per layer type (reading Q13) on the first 4 blocks of the Llama-3-8B shapes."""
    _need_gpu(40)
    spec = I.llama3_8b_spec(n_blocks=4, schedule=True)
    plan, worst, n = _run_config_step(spec, 128, 2048, 64, 6)
    assert plan.n_buckets == 3


@pytest.mark.parametrize("T", [16, 32, 64, 128, 256])
def test_config3_sweep_sampled(T):
    """BASELINE configs[2]: Phi_{K,T} on the 4096 x 11008 row-scaled Gaussian matrix, sampled tiles."""
    _need_gpu()
    H, W = 4096, 11008
    G = I.row_scaled_gaussian(H, W, seed_cfg=2, layer_index=1, dtype=torch.bfloat16, device=DEV)
    U = torch.full_like(G, float("nan"))
    hp = hm.HParams(K=5, eps=1e-7)
    plan = hm.Plan.from_tensors([U], [G], None, T).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    rng = np.random.default_rng(7 + T)
    ohp = PU.oracle_hp(hp)
    worst = 0.0
    for _ in range(64):
        r, c = int(rng.integers(H // T)), int(rng.integers(W // T))
        g = PU.f64(_cut(G, T, r, c))
        ref = PU.O.phi(g, ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
        e = np.linalg.norm(PU.f64(_cut(U, T, r, c)) - ref) / np.linalg.norm(ref)
        worst = max(worst, e)
    assert worst <= PU.TOL_TC, f"T={T}: worst sampled tile error {worst:.3e}"
    assert bool(torch.isfinite(U.float()).all())


@pytest.mark.parametrize("T", [16, 32, 64, 128, 256, 512])
def test_step_is_deterministic_at_scale(T):
    """The same step from the same bits twice: bitwise identical W' and M' (no race between the tiles in flight,
    the prefetches and the stores; fixed summation orders).  GPT-2-XL shapes: ragged at every T >= 128."""
    _need_gpu(40)
    spec = I.gpt2_xl_spec(n_blocks=4)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    outs = []
    for rep in range(2):
        Ws, Gs, Ms = [], [], []
        for i in range(len(spec.layers)):
            W, G, M = I.make_layer_tensors(spec, i, dtype=torch.bfloat16, device=DEV)
            Ws.append(W); Gs.append(G); Ms.append(M)
        plan = hm.Plan.from_tensors(Ws, Gs, Ms, T, workspace_cap_bytes=1024 << 20).bind()
        plan.step(hp)
        plan.step(hp)                      # second step on the updated state
        torch.cuda.synchronize()
        outs.append((Ws, Ms))
        plan.destroy()
    for a, b in zip(outs[0][0] + outs[0][1], outs[1][0] + outs[1][1]):
        assert torch.equal(a, b)
        assert bool(torch.isfinite(a.float()).all())
