"""GPU parity tests of the T = 256 kernel (one tile per CTA pair, tcgen05 cta_group::2,
csrc/kernels_tc256.cu) against the float64 oracle."""
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
    return I.lowrank_plus_noise(H, W, 32, seed_cfg=seed, layer_index=0, tensor_id=I.TENSOR_G)


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
def test_tc256_phi(K, kind):
    _need_gpu()
    G = _inputs(512, 768, 61, kind)                 # 2 x 3 tiles
    hp = hm.HParams(K=K, eps=1e-7)
    U = _run_phi(G, 256, hp)
    if K == 0:
        ref = PU.O.phi_tiled(PU.f64(G), 256, 0, eps=float(np.float32(1e-7)))
        d = np.abs(PU.f64(U) - ref)
        assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-12)
    else:
        PU.check_phi(U, G, 256, hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("H,W", [(256, 256), (300, 520), (100, 264), (257, 128)])
def test_tc256_ragged_phi(H, W):
    """Edge tiles (including tiles whose lower CTA half is entirely padding); canaries untouched."""
    _need_gpu()
    ld = ((W + 7) // 8) * 8 + 16
    Gfull = torch.zeros(H, ld, dtype=torch.bfloat16)
    Gfull[:, :W] = _inputs(H, W, 62)
    Gd = Gfull.to(DEV)
    Ud = torch.full((H + 3, ld), 7.0, dtype=torch.bfloat16, device=DEV)
    hp = hm.HParams(K=5, eps=1e-7)
    plan = hm.Plan.from_tensors([Ud[:H, :W]], [Gd[:, :W]], None, 256).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    U = Ud.cpu()
    assert torch.all(U[:H, W:] == 7.0) and torch.all(U[H:] == 7.0), "wrote outside H x W"
    PU.check_phi(U[:H, :W], Gfull[:, :W], 256, hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("nesterov,wd", [(True, 0.01), (False, 0.0)])
def test_tc256_step(nesterov, wd):
    _need_gpu()
    shapes = [(512, 256), (256, 768), (300, 264)]
    Ws, Gs, Ms = [], [], []
    for i, (h, w) in enumerate(shapes):
        Gs.append(I.lowrank_plus_noise(h, w, 32, seed_cfg=63, layer_index=i, tensor_id=I.TENSOR_G))
        Ms.append(I.lowrank_plus_noise(h, w, 32, seed_cfg=63, layer_index=i, tensor_id=I.TENSOR_M))
        Ws.append(I.gaussian(h, w, seed_cfg=63, layer_index=i, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02))
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=nesterov, lr=0.02, wd=wd, scale_c=0.2)
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    plan = hm.Plan.from_tensors(Wd, Gd, Md, 256).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        PU.check_step(Ws[i], Gs[i], Ms[i], Wd[i].cpu(), Md[i].cpu(), 256, hp, PU.TOL_TC, storage_bf16=True)
        assert torch.equal(Gd[i].cpu(), Gs[i])


def test_tc256_one_hot_positions():
    _need_gpu()
    H, W, T = 520, 304, 256
    G = torch.zeros(H, W, dtype=torch.bfloat16)
    want = torch.zeros_like(G)
    for r in range((H + T - 1) // T):
        for c in range((W + T - 1) // T):
            i = min(r * T + (137 * r + 11 * c + 130) % T, H - 1)
            j = min(c * T + (53 * c + 29 * r + 70) % T, W - 1)
            G[i, j] = 2.0 + r + c
            want[i, j] = 1.0
    U = _run_phi(G, T, hm.HParams(K=0, eps=0.0))
    assert torch.equal(U, want)


def test_ns_tiles_bf16_256():
    _need_gpu()
    tiles = torch.stack([_inputs(256, 256, 64 + i, "gauss") for i in range(3)])
    out = hm.himuon_ns_tiles(tiles.to(DEV), K=5, eps=1e-7).cpu()
    ohp = PU.oracle_hp(hm.HParams(K=5, eps=1e-7))
    for i in range(3):
        ref = PU.O.phi(PU.f64(tiles[i]), ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
        e = np.linalg.norm(PU.f64(out[i]) - ref) / np.linalg.norm(ref)
        assert e <= PU.TOL_TC, f"tile {i}: {e:.3e}"


def test_t256_width_not_multiple_of_8_runs_on_the_large_tile_path():
    """bf16 widths that are not a multiple of 8 have no TMA path at T = 256: served by the large-tile (cuBLAS) path."""
    _need_gpu()
    G = _inputs(300, 300, 65)
    hp = hm.HParams(K=5, eps=1e-7)
    U = _run_phi(G, 256, hp)
    PU.check_phi(U, G, 256, hp, PU.TOL_TC, out_is_bf16=True)
