"""GPU parity tests of the T = 64 tensor-core kernel (two 64 x 64 tiles stacked per tcgen05 MMA,
csrc/kernels_tc64.cu) against the float64 oracle, and of the mixed-T plans that use it."""
import numpy as np
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm
import parity_util as PU

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def _inputs(H, W, seed, kind="lowrank"):
    if kind == "gauss":
        return I.row_scaled_gaussian(H, W, seed_cfg=seed, dtype=torch.bfloat16)
    return I.lowrank_plus_noise(H, W, 16, seed_cfg=seed, layer_index=0, tensor_id=I.TENSOR_G)


def _run_phi(G, T, hp):
    Gd = G.to(DEV)
    Ud = torch.full_like(Gd, float("nan"))
    plan = hm.Plan.from_tensors([Ud], [Gd], None, T).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    plan.destroy()
    return Ud.cpu()


@pytest.mark.parametrize("K", [0, 1, 5])
@pytest.mark.parametrize("kind", ["gauss", "lowrank"])
def test_tc64_phi(K, kind):
    _need_gpu()
    G = _inputs(256, 320, 41, kind)                  # 4 x 5 = 20 tiles -> 10 super-tiles over several CTAs
    hp = hm.HParams(K=K, eps=1e-7)
    U = _run_phi(G, 64, hp)
    if K == 0:
        ref = PU.O.phi_tiled(PU.f64(G), 64, 0, eps=float(np.float32(1e-7)))
        d = np.abs(PU.f64(U) - ref)
        assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-12)
    else:
        PU.check_phi(U, G, 64, hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("H,W", [(64, 64), (192, 64), (100, 136), (65, 200), (1600 // 8, 72)])
def test_tc64_ragged_and_odd_counts(H, W):
    """Odd tile counts (the last super-tile holds one tile), edge tiles, gutter and rows past H untouched."""
    _need_gpu()
    ld = ((W + 7) // 8) * 8 + 16
    Gfull = torch.zeros(H, ld, dtype=torch.bfloat16)
    Gfull[:, :W] = _inputs(H, W, 42)
    Gd = Gfull.to(DEV)
    Ud = torch.full((H + 3, ld), 7.0, dtype=torch.bfloat16, device=DEV)
    hp = hm.HParams(K=5, eps=1e-7)
    plan = hm.Plan.from_tensors([Ud[:H, :W]], [Gd[:, :W]], None, 64).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    U = Ud.cpu()
    assert torch.all(U[:H, W:] == 7.0) and torch.all(U[H:] == 7.0), "wrote outside H x W"
    PU.check_phi(U[:H, :W], Gfull[:, :W], 64, hp, PU.TOL_TC, out_is_bf16=True)


def _param_set(shapes, seed, rank=16):
    Ws, Gs, Ms = [], [], []
    for i, (h, w) in enumerate(shapes):
        Gs.append(I.lowrank_plus_noise(h, w, rank, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_G))
        Ms.append(I.lowrank_plus_noise(h, w, rank, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_M))
        Ws.append(I.gaussian(h, w, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02))
    return Ws, Gs, Ms


@pytest.mark.parametrize("nesterov,wd", [(True, 0.01), (False, 0.0)])
def test_tc64_step_cross_layer_supertiles(nesterov, wd):
    """Layers with odd tile counts: super-tiles pair tiles of DIFFERENT layers (tau, maps per tile)."""
    _need_gpu()
    shapes = [(64, 192), (128, 64), (100, 72), (192, 192)]          # 3, 2, 4, 9 tiles
    Ws, Gs, Ms = _param_set(shapes, 43)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=nesterov, lr=0.02, wd=wd, scale_c=0.2)
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    plan = hm.Plan.from_tensors(Wd, Gd, Md, 64).bind()
    assert plan.n_buckets == 1
    plan.step(hp)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        PU.check_step(Ws[i], Gs[i], Ms[i], Wd[i].cpu(), Md[i].cpu(), 64, hp, PU.TOL_TC, storage_bf16=True)
        assert torch.equal(Gd[i].cpu(), Gs[i])


def test_mixed_T_schedule_step():
    """Runtime tile schedule per layer (reading Q13): buckets T = 64 and T = 128 in one plan, one step."""
    _need_gpu()
    shapes = [(128, 256), (256, 256), (64, 256), (256, 128)]
    Tl = [64, 128, 64, 128]
    Ws, Gs, Ms = _param_set(shapes, 44)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    plan = hm.Plan.from_tensors(Wd, Gd, Md, 128, T_per_layer=Tl).bind()
    assert plan.n_buckets == 2
    plan.step(hp)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        PU.check_step(Ws[i], Gs[i], Ms[i], Wd[i].cpu(), Md[i].cpu(), Tl[i], hp, PU.TOL_TC, storage_bf16=True)


@pytest.mark.parametrize("T,n", [(64, 7), (128, 5)])
def test_ns_tiles_bf16(T, n):
    """himuon_ns_tiles on packed [n, T, T] bf16 tiles (the paper's Fig. 7 workload)."""
    _need_gpu()
    tiles = torch.stack([_inputs(T, T, 45 + i) for i in range(n)])
    hp = hm.HParams(K=5, eps=1e-7)
    out = hm.himuon_ns_tiles(tiles.to(DEV), K=5, eps=1e-7).cpu()
    ohp = PU.oracle_hp(hp)
    for i in range(n):
        ref = PU.O.phi(PU.f64(tiles[i]), ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
        e = np.linalg.norm(PU.f64(out[i]) - ref) / np.linalg.norm(ref)
        assert e <= PU.TOL_TC, f"tile {i}: {e:.3e}"


def test_tc64_indexing_bit_exact():
    """K = 0 on integer-tagged inputs with a one-hot structure per tile: positions come back exactly."""
    _need_gpu()
    H, W = 192, 136
    G = torch.zeros(H, W, dtype=torch.bfloat16)
    for r in range(0, H, 64):
        for c in range(0, W, 64):
            i, j = (r // 64 * 7 + c // 64 * 3) % min(64, H - r), (r // 64 * 5 + c // 64 * 11) % min(64, W - c)
            G[r + i, c + j] = 2.0
    U = _run_phi(G, 64, hm.HParams(K=0, eps=0.0))
    assert torch.equal(U, (G != 0).to(torch.bfloat16)), "one-hot positions moved"
