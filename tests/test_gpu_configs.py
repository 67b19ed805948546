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


# ---- W0 = 0: the update IS the map.  W' = -lr tau U with one RNE rounding, so U_gpu = -W'/(lr tau) is recovered
# (to 2^-9 per element) and the north-star bar - per-tile relative Frobenius error <= 3e-2 against the float64 oracle -
# is applied to it DIRECTLY, at full size, in the launch bench.py times.  Beside the oracle-checked tiles (every tile
# of one layer of each shape + a seeded sample of the rest) EVERY tile is checked for finiteness and
# against the fp32-arithmetic kernel (HIMUON_PATH_FP32, itself oracle-pinned to 1e-4) on the GPU.

def _bits(t):
    """bf16 tensor -> uint16 numpy bit patterns (host)."""
    return t.contiguous().cpu().view(torch.int16).numpy().view(np.uint16)


def _gather_tiles(x, T, rc):
    """Tiles (r, c) of a 2-D device tensor as a packed [n, T, T] host array of bf16 bits, zero-padded (B_T)."""
    H, W = x.shape
    R, C = -(-H // T), -(-W // T)
    if R * T != H or C * T != W:
        x = torch.nn.functional.pad(x, (0, C * T - W, 0, R * T - H))
    t4 = x.view(R, T, C, T).permute(0, 2, 1, 3)           # [R, C, T, T] view
    r = torch.tensor([a for a, _ in rc], device=x.device)
    c = torch.tensor([b for _, b in rc], device=x.device)
    return _bits(t4[r, c])


def _per_tile_rel_err_gpu(Ua, Ub, T):
    """max over the tiles of ||Ua - Ub||_F / ||Ub||_F, on the device (tiles with Ub = 0 must have Ua = 0)."""
    H, W = Ua.shape
    R, C = -(-H // T), -(-W // T)
    d, b = (Ua.float() - Ub.float()), Ub.float()
    if R * T != H or C * T != W:
        d = torch.nn.functional.pad(d, (0, C * T - W, 0, R * T - H))
        b = torch.nn.functional.pad(b, (0, C * T - W, 0, R * T - H))
    num = (d.view(R, T, C, T) ** 2).sum(dim=(1, 3))
    den = (b.view(R, T, C, T) ** 2).sum(dim=(1, 3))
    err = torch.where(den > 0, torch.sqrt(num / den.clamp_min(1e-38)), torch.sqrt(num))
    return float(err.max())


def _run_config_w0(spec, T_default, cap_mb, frac, seed, whole_layers, path=hm.HIMUON_PATH_AUTO, tol=PU.TOL_TC,
                   crosscheck=True):
    import oracle_pool as OP
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    Tl = [l.T or T_default for l in spec.layers]
    n_layers = len(spec.layers)
    Ws, Gs, Ms = [], [], []
    for i in range(n_layers):
        W, G, M = I.make_layer_tensors(spec, i, dtype=torch.bfloat16, device=DEV)
        Ws.append(torch.zeros_like(W)); Gs.append(G); Ms.append(M)
    # tiles the oracle sees: every tile of the first layer of each (H, W, T), a seeded fraction of all the others
    rng = np.random.default_rng(seed)
    picks, seen = {}, set()
    for li, l in enumerate(spec.layers):
        T = Tl[li]
        R, C = -(-l.H // T), -(-l.W // T)
        if whole_layers and (l.H, l.W, T) not in seen:
            seen.add((l.H, l.W, T))
            picks[li] = [(r, c) for r in range(R) for c in range(C)]
        else:
            n = rng.binomial(R * C, frac)
            flat = rng.choice(R * C, size=n, replace=False) if n else []
            picks[li] = sorted({(R - 1, C - 1)} | {(int(f) // C, int(f) % C) for f in flat})   # + the corner tile
    G_t = {li: _gather_tiles(Gs[li], Tl[li], rc) for li, rc in picks.items()}
    M0_t = {li: _gather_tiles(Ms[li], Tl[li], rc) for li, rc in picks.items()}
    if crosscheck:                                            # the same step with fp32 arithmetic, from the same bits
        Wb = [torch.zeros_like(w) for w in Ws]
        Mb = [m.clone() for m in Ms]
    plan = hm.Plan.from_tensors(Ws, Gs, Ms, T_default, T_per_layer=Tl if any(l.T for l in spec.layers) else None,
                                path=path, workspace_cap_bytes=cap_mb << 20).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    # (1) every tile: finite
    for li in range(n_layers):
        assert bool(torch.isfinite(Ws[li].float()).all()) and bool(torch.isfinite(Ms[li].float()).all()), f"layer {li}: non-finite"
    # (2) every tile: against the fp32-arithmetic kernel on the same bits (M' bitwise: same fp32 formula, one RNE)
    worst_x = 0.0
    if crosscheck:
        pb = hm.Plan.from_tensors(Wb, Gs, Mb, T_default, T_per_layer=Tl if any(l.T for l in spec.layers) else None,
                                  path=hm.HIMUON_PATH_FP32, workspace_cap_bytes=cap_mb << 20).bind()
        pb.step(hp)
        torch.cuda.synchronize()
        for li in range(n_layers):
            assert torch.equal(Ms[li], Mb[li]), f"layer {li}: M' differs between the bf16 and the fp32 kernel"
            worst_x = max(worst_x, _per_tile_rel_err_gpu(Ws[li], Wb[li], Tl[li]))   # U = -W'/(lr tau): the scale cancels
        # ||U_bf - U_oracle|| <= ||U_bf - U_fp32|| + ||U_fp32 - U_oracle||, and the fp32 kernel's stored result is within
        # 1e-4 (arithmetic, oracle-pinned) + 2^-9/sqrt(3) = 1.1e-3 (its one bf16 output rounding) of the oracle
        assert worst_x <= tol - 1.2e-3, f"worst tile of all {plan.n_tiles}: bf16 vs fp32 kernel {worst_x:.3e}"
        pb.destroy()
        del Wb, Mb
    # (3) the oracle-checked tiles, at the north-star tolerance on U itself
    ohp = PU.oracle_hp(hp)
    hpd = dict(lr=ohp.lr, beta=ohp.beta, nesterov=ohp.nesterov, wd=ohp.wd, K=ohp.K, a=ohp.a, b=ohp.b, c=ohp.c,
               eps=ohp.eps, scale_c=ohp.scale_c)
    n_checked, worst_u, worst_m = 0, 0.0, 0.0
    for T in sorted(set(Tl)):
        tiles = []
        for li, rc in picks.items():
            if Tl[li] != T or not rc:
                continue
            W1, M1 = _gather_tiles(Ws[li], T, rc), _gather_tiles(Ms[li], T, rc)
            tiles += [(G_t[li][k], M0_t[li][k], W1[k], M1[k]) for k in range(len(rc))]
        res = OP.check_tiles_w0(hpd, T, PU.O.tau(4 * T, 4 * T, T, ohp.scale_c), tiles)
        assert np.all(res[:, 2] == 1.0), "non-finite output tile"
        n_checked += len(tiles)
        worst_u, worst_m = max(worst_u, float(res[:, 0].max())), max(worst_m, float(res[:, 1].max()))
    assert worst_m <= 1.0, f"M' off by {worst_m:.3f} x its allowance (one bf16 ulp + fp32 slack)"
    assert worst_u <= tol, f"worst per-tile rel Fro error of U over {n_checked} oracle-checked tiles: {worst_u:.3e} > {tol}"
    print(f"{spec.name} T={T_default}: {n_checked} tiles vs oracle, worst U err {worst_u:.3e}, M' ratio {worst_m:.3f}; "
          f"all {plan.n_tiles} tiles vs fp32 kernel: {worst_x:.3e}")
    return plan, n_checked, worst_u


def test_config2_gpt2_small_every_tile_w0():
    """BASELINE configs[1]: every one of the 5184 tiles against the oracle, U recovered from a W0 = 0 step."""
    _need_gpu()
    plan, n, worst = _run_config_w0(I.gpt2_small_spec(), 128, 2048, 1.0, 12, whole_layers=True)
    assert plan.n_tiles == 5184 and n >= 5184


def test_config4_gpt2_xl_whole_layers_and_sample_w0():
    """BASELINE configs[3] (ragged, 256 MB cap): every tile of one layer of each shape + a 2 % sample vs the oracle;
    every tile finite and within tolerance of the fp32 kernel."""
    _need_gpu(40)
    plan, n, worst = _run_config_w0(I.gpt2_xl_spec(), 128, 256, 0.02, 14, whole_layers=True)
    assert plan.n_tiles == 94848 and n >= 169 + 650 + 650 + 1500


def test_config5_llama3_8b_whole_layers_and_sample_w0():
    """BASELINE configs[4] at T = 128, the launch bench.py times: every tile of one layer of each of the four shapes
    (8448 tiles) + a 2 % sample of the other 417 536 vs the oracle at 3e-2 on U; all 425 984 tiles finite and within
    tolerance of the fp32 kernel."""
    _need_gpu(120)
    plan, n, worst = _run_config_w0(I.llama3_8b_spec(), 128, 2048, 0.02, 15, whole_layers=True)
    assert plan.n_tiles == 425984 and n >= 8448 + 7500


@pytest.mark.parametrize("T,frac", [(64, 0.02), (256, 0.02), (32, 0.002), (16, 0.0005)])
def test_config5_llama3_8b_other_tile_sizes_w0(T, frac):
    """The same parameter set at the other tile sizes: a seeded sample vs the oracle (smaller fractions where the
    tile count is in the millions), every tile vs the fp32 kernel where that kernel exists (T <= 128)."""
    _need_gpu(120)
    plan, n, worst = _run_config_w0(I.llama3_8b_spec(), T, 2048, frac, 16 + T, whole_layers=False, crosscheck=T <= 128)
    assert n >= 1000


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
