"""GPU parity tests of the large-tile path (csrc/kernels_gemm.cu): T = 512 tiles and the full-matrix branch
T >= max(H, W) beyond 256 (the paper's T = infinity warm start and its T = 512 default, PAPER.md:135-138, :243-249,
:386), whose products run on cuBLAS.  Tolerances: bf16 storage (TF32 products) 3e-2, fp32 storage 1e-4."""
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


def _run_phi(G, T, hp, path=hm.HIMUON_PATH_AUTO):
    Gd = G.to(DEV)
    Ud = torch.full_like(Gd, float("nan"))
    plan = hm.Plan.from_tensors([Ud], [Gd], None, T, path=path).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    plan.destroy()
    return Ud.cpu()


@pytest.mark.parametrize("H,W,T", [(1024, 1536, 512), (700, 520, 512), (640, 384, 100000), (300, 900, 1024), (512, 512, 512)])
def test_large_tiles_phi_bf16(H, W, T):
    _need_gpu()
    G = I.lowrank_plus_noise(H, W, 32, seed_cfg=71, layer_index=0, tensor_id=I.TENSOR_G)
    hp = hm.HParams(K=5, eps=1e-7)
    U = _run_phi(G, T, hp)
    PU.check_phi(U, G, T, hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("H,W,T", [(600, 400, 1024), (512, 768, 256), (520, 1030, 512)])
def test_large_tiles_phi_fp32(H, W, T):
    """fp32 storage: true fp32 products, the <= 1e-4 path (also T = 256 on fp32 storage)."""
    _need_gpu()
    G = I.gaussian(H, W, seed_cfg=72, dtype=torch.float32)
    hp = hm.HParams(K=5, eps=1e-7)
    U = _run_phi(G, T, hp)
    PU.check_phi(U, G, T, hp, PU.TOL_FP32, out_is_bf16=False)


@pytest.mark.parametrize("nesterov", [True, False])
def test_full_to_local_schedule_step(nesterov):
    """One step each of the paper's schedule infinity -> 512 -> 128 on the same parameters; momentum buffers are
    plan-independent and survive re-planning."""
    _need_gpu()
    shapes = [(768, 1024), (1024, 520)]
    Ws, Gs, Ms = [], [], []
    for i, (h, w) in enumerate(shapes):
        Gs.append(I.lowrank_plus_noise(h, w, 32, seed_cfg=73, layer_index=i, tensor_id=I.TENSOR_G))
        Ms.append(I.lowrank_plus_noise(h, w, 32, seed_cfg=73, layer_index=i, tensor_id=I.TENSOR_M))
        Ws.append(I.gaussian(h, w, seed_cfg=73, layer_index=i, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02))
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=nesterov, lr=0.02, wd=0.01, scale_c=0.2)
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    Wh, Mh = [w.clone() for w in Ws], [m.clone() for m in Ms]
    for T in (1 << 20, 512, 128):
        plan = hm.Plan.from_tensors(Wd, Gd, Md, T).bind()
        plan.step(hp)
        torch.cuda.synchronize()
        plan.destroy()
        for i in range(len(shapes)):
            PU.check_step(Wh[i], Gs[i], Mh[i], Wd[i].cpu(), Md[i].cpu(), T, hp, PU.TOL_TC, storage_bf16=True)
            Wh[i], Mh[i] = Wd[i].cpu(), Md[i].cpu()          # continue from what the GPU stored


def test_ns_tiles_512():
    _need_gpu()
    tiles = torch.stack([I.row_scaled_gaussian(512, 512, seed_cfg=74 + i, dtype=torch.bfloat16) for i in range(2)])
    out = hm.himuon_ns_tiles(tiles.to(DEV), K=5, eps=1e-7).cpu()
    ohp = PU.oracle_hp(hm.HParams(K=5, eps=1e-7))
    for i in range(2):
        ref = PU.O.phi(PU.f64(tiles[i]), ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
        e = np.linalg.norm(PU.f64(out[i]) - ref) / np.linalg.norm(ref)
        assert e <= PU.TOL_TC, f"tile {i}: {e:.3e}"


def _rect_err(U, ref, Th, Tw):
    H, W = ref.shape
    worst = 0.0
    for r in range(-(-H // Th)):
        for c in range(-(-W // Tw)):
            a, b = U[r * Th:(r + 1) * Th, c * Tw:(c + 1) * Tw], ref[r * Th:(r + 1) * Th, c * Tw:(c + 1) * Tw]
            worst = max(worst, np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-30))
    return worst


@pytest.mark.parametrize("H,W,Th,Tw", [(256, 512, 64, 256), (300, 500, 128, 32), (1024, 256, 16, 256), (200, 200, 256, 64)])
def test_rectangular_tiles_phi(H, W, Th, Tw):
    """Rectangular tiles (T_h, T_w) of the tile-shape study against phi_tiled_rect."""
    _need_gpu()
    G = I.lowrank_plus_noise(H, W, 32, seed_cfg=75, layer_index=0, tensor_id=I.TENSOR_G)
    Gd = G.to(DEV)
    Ud = torch.full_like(Gd, float("nan"))
    hp = hm.HParams(K=5, eps=1e-7)
    plan = hm.Plan.from_tensors([Ud], [Gd], None, Th, Tw_per_layer=[Tw]).bind()
    assert plan.n_tiles == -(-H // Th) * -(-W // Tw)
    plan.phi(hp)
    torch.cuda.synchronize()
    ohp = PU.oracle_hp(hp)
    ref = PU.O.phi_tiled_rect(PU.f64(G), Th, Tw, ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
    assert _rect_err(PU.f64(Ud.cpu()), ref, Th, Tw) <= PU.TOL_TC


def test_rectangular_tiles_step():
    """Full step with rectangular tiles: tau = c sqrt(max(T_h, T_w))."""
    _need_gpu()
    H, W, Th, Tw = 384, 320, 128, 64
    G = I.lowrank_plus_noise(H, W, 32, seed_cfg=76, layer_index=0, tensor_id=I.TENSOR_G)
    M = I.lowrank_plus_noise(H, W, 32, seed_cfg=76, layer_index=0, tensor_id=I.TENSOR_M)
    W0 = I.gaussian(H, W, seed_cfg=76, layer_index=0, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    Wd, Gd, Md = W0.to(DEV), G.to(DEV), M.to(DEV)
    plan = hm.Plan.from_tensors([Wd], [Gd], [Md], Th, Tw_per_layer=[Tw]).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    Wr, Mr, Ur = PU.O.step_rect(PU.f64(W0), PU.f64(G), PU.f64(M), PU.oracle_hp(hp), Th, Tw)
    m_gpu, w_gpu = PU.f64(Md.cpu()), PU.f64(Wd.cpu())
    assert np.all(np.abs(m_gpu - Mr) <= PU.BF16_ULP * np.abs(Mr) + 2.0 ** -21 * (np.abs(0.95 * PU.f64(M)) + np.abs(PU.f64(G))) + 1e-30)
    tau = PU.O.tau_rect(H, W, Th, Tw, 0.2)
    for r in range(H // Th):
        for c in range(W // Tw):
            sl = (slice(r * Th, (r + 1) * Th), slice(c * Tw, (c + 1) * Tw))
            dW = np.linalg.norm(w_gpu[sl] - Wr[sl])
            bound = PU.BF16_ULP * np.linalg.norm(Wr[sl]) + 0.02 * tau * PU.TOL_TC * np.linalg.norm(Ur[sl])
            assert dW <= bound, f"tile ({r},{c}): {dW / bound:.3f}"


@pytest.mark.parametrize("H,W", [(1024, 3072), (2560, 1032)])
def test_full_matrix_branch_on_the_cta_pair_gemm(H, W):
    """Full-matrix branch on shapes whose contractions are longer than 512, i.e. the CTA-pair (cta_group::2) form of
    the large-tile GEMM in all three products, wide and tall (transposed iterate), with a ragged last row
    block: against the oracle's full-matrix Phi_K and, run twice from the same bits, bitwise identical."""
    _need_gpu()
    G = I.lowrank_plus_noise(H, W, 64, seed_cfg=77, layer_index=0, tensor_id=I.TENSOR_G)
    hp = hm.HParams(K=5, eps=1e-7)
    U1 = _run_phi(G, 1 << 20, hp)
    U2 = _run_phi(G, 1 << 20, hp)
    assert torch.equal(U1, U2)
    PU.check_phi(U1, G, max(H, W), hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("H,W", [(1100, 1536), (2056, 1000)])
def test_full_matrix_step_on_big_tiles(H, W):
    """Full step (momentum, Nesterov, weight decay) on matrices of more than 1 M elements, wide and tall: the fused ends of
    big tiles run on their own grid, tall ones through the shared-memory transposes (lt_prep_t / lt_update_t), here with
    ragged last patches in both directions; two steps, the second from the stored state of the first."""
    _need_gpu()
    G = I.lowrank_plus_noise(H, W, 48, seed_cfg=78, layer_index=0, tensor_id=I.TENSOR_G)
    M0 = I.lowrank_plus_noise(H, W, 48, seed_cfg=78, layer_index=0, tensor_id=I.TENSOR_M)
    W0 = I.gaussian(H, W, seed_cfg=78, layer_index=0, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    Wd, Gd, Md = W0.to(DEV), G.to(DEV), M0.to(DEV)
    Wh, Mh = W0, M0
    plan = hm.Plan.from_tensors([Wd], [Gd], [Md], 1 << 20).bind()
    for _ in range(2):
        plan.step(hp)
        torch.cuda.synchronize()
        PU.check_step(Wh, G, Mh, Wd.cpu(), Md.cpu(), 1 << 20, hp, PU.TOL_TC, storage_bf16=True)
        Wh, Mh = Wd.cpu(), Md.cpu()
    plan.destroy()
