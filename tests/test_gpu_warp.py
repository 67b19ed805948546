"""GPU parity tests of the warp-level mma.sync kernel (T = 16 and T = 32, bf16 storage,
csrc/kernels_warp.cu) against the float64 oracle."""
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


@pytest.mark.parametrize("T", [16, 32])
@pytest.mark.parametrize("K", [0, 1, 5])
@pytest.mark.parametrize("kind", ["gauss", "lowrank"])
def test_warp_phi(T, K, kind):
    _need_gpu()
    G = _inputs(512, 1024, 51, kind)              # 2048 / 512 tiles: several waves of warps
    hp = hm.HParams(K=K, eps=1e-7)
    U = _run_phi(G, T, hp)
    if K == 0:
        ref = PU.O.phi_tiled(PU.f64(G), T, 0, eps=float(np.float32(1e-7)))
        d = np.abs(PU.f64(U) - ref)
        assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-12)
    else:
        PU.check_phi(U, G, T, hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("T", [16, 32])
@pytest.mark.parametrize("H,W,pad", [(33, 47, 1), (100, 150, 2), (16, 16, 0), (70, 31, 3)])
def test_warp_ragged_odd_widths(T, H, W, pad):
    """Edge tiles, odd widths and odd leading dimensions (16-bit access path); canaries untouched."""
    _need_gpu()
    ld = W + pad
    Gfull = torch.zeros(H, ld, dtype=torch.bfloat16)
    Gfull[:, :W] = _inputs(H, W, 52)
    Gd = Gfull.to(DEV)
    Ud = torch.full((H + 2, ld), 7.0, dtype=torch.bfloat16, device=DEV)
    hp = hm.HParams(K=5, eps=1e-7)
    plan = hm.Plan.from_tensors([Ud[:H, :W]], [Gd[:, :W]], None, T).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    U = Ud.cpu()
    assert torch.all(U[:H, W:] == 7.0) and torch.all(U[H:] == 7.0), "wrote outside H x W"
    PU.check_phi(U[:H, :W], Gfull[:, :W], T, hp, PU.TOL_TC, out_is_bf16=True)


def _param_set(shapes, seed, rank=16):
    Ws, Gs, Ms = [], [], []
    for i, (h, w) in enumerate(shapes):
        Gs.append(I.lowrank_plus_noise(h, w, rank, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_G))
        Ms.append(I.lowrank_plus_noise(h, w, rank, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_M))
        Ws.append(I.gaussian(h, w, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02))
    return Ws, Gs, Ms


@pytest.mark.parametrize("T", [16, 32])
@pytest.mark.parametrize("nesterov,wd", [(True, 0.01), (False, 0.0)])
def test_warp_step(T, nesterov, wd):
    _need_gpu()
    shapes = [(64, 96), (48, 40), (100, 72), (32, 160)]
    Ws, Gs, Ms = _param_set(shapes, 53)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=nesterov, lr=0.02, wd=wd, scale_c=0.2)
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    plan = hm.Plan.from_tensors(Wd, Gd, Md, T).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        PU.check_step(Ws[i], Gs[i], Ms[i], Wd[i].cpu(), Md[i].cpu(), T, hp, PU.TOL_TC, storage_bf16=True)
        assert torch.equal(Gd[i].cpu(), Gs[i])


@pytest.mark.parametrize("T", [16, 32])
def test_warp_one_hot_positions(T):
    """K = 0 on tiles holding a single non-zero: output non-zero exactly there (bit-exact indexing)."""
    _need_gpu()
    H, W = 75, 110
    G = torch.zeros(H, W, dtype=torch.bfloat16)
    want = torch.zeros_like(G)
    for r in range((H + T - 1) // T):
        for c in range((W + T - 1) // T):
            i = min(r * T + (5 * r + 11 * c) % T, H - 1)
            j = min(c * T + (7 * c + 3 * r) % T, W - 1)
            G[i, j] = 2.0 + r
            want[i, j] = 1.0
    U = _run_phi(G, T, hm.HParams(K=0, eps=0.0))
    assert torch.equal(U, want)


@pytest.mark.parametrize("T,n", [(16, 37), (32, 9)])
def test_ns_tiles_bf16_small_T(T, n):
    _need_gpu()
    tiles = torch.stack([_inputs(T, T, 54 + i, "gauss") for i in range(n)])
    out = hm.himuon_ns_tiles(tiles.to(DEV), K=5, eps=1e-7).cpu()
    ohp = PU.oracle_hp(hm.HParams(K=5, eps=1e-7))
    for i in range(n):
        ref = PU.O.phi(PU.f64(tiles[i]), ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
        e = np.linalg.norm(PU.f64(out[i]) - ref) / np.linalg.norm(ref)
        assert e <= PU.TOL_TC, f"tile {i}: {e:.3e}"
