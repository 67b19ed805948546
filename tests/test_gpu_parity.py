"""GPU parity tests: the CUDA path (through the C-ABI) against the float64 oracle, element by
element / tile by tile on the same seeded bits.  Run with `-m gpu` on a B200."""
import numpy as np
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm
from paper_2606_27216_b200 import binding as B
import parity_util as PU

pytestmark = pytest.mark.gpu

DEV = "cuda"


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def run_phi(G: torch.Tensor, T: int, hp, path=hm.HIMUON_PATH_AUTO, cap=0):
    Gd = G.to(DEV)
    Ud = torch.full_like(Gd, float("nan"))
    plan = hm.Plan.from_tensors([Ud], [Gd], None, T, path=path, workspace_cap_bytes=cap).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    plan.destroy()
    return Ud.cpu()


# ----------------------------------------------------------------------------- fp32 path

@pytest.mark.parametrize("T", [32, 128])
def test_fp32_path_cubic_iteration_c_zero(T):
    """(a, b, c) = (1.5, -0.5, 0), the cubic Newton-Schulz iteration: c = 0 is served by the fp32 kernel (<= 1e-4 against
    the oracle) and refused by the bf16 tensor-core kernels, which iterate on c^(1/4) X (include/himuon.h)."""
    _need_gpu()
    G = I.gaussian(2 * T + 8, 3 * T, seed_cfg=0, layer_index=5, dtype=torch.float32)
    hp = hm.HParams(K=5, a=1.5, b=-0.5, c=0.0, eps=1e-7)
    U = run_phi(G, T, hp)
    PU.check_phi(U, G, T, hp, PU.TOL_FP32, out_is_bf16=False)
    Gb = G.to(torch.bfloat16)
    if T >= 64:
        with pytest.raises(hm.HimuonError) as ei:
            run_phi(Gb, T, hp)
        assert ei.value.status == B.HIMUON_ERR_UNSUPPORTED
    else:                                                               # warp kernel: plain state, any (a, b, c)
        PU.check_phi(run_phi(Gb, T, hp), Gb, T, hp, PU.TOL_TC, out_is_bf16=True)
    Ub = run_phi(Gb, T, hp, path=hm.HIMUON_PATH_FP32)                  # bf16 storage, fp32 arithmetic: accepted
    PU.check_phi(Ub, Gb, T, hp, 5e-3, out_is_bf16=True)               # one bf16 rounding of the output


@pytest.mark.parametrize("T", [16, 32, 64, 128])
def test_config1_fp32_phi(T):
    """BASELINE config 1: fp32 256x512 N(0,1) seed 0, K=5, eps=1e-7 (T=64 -> 32 tiles, reading Q1)."""
    _need_gpu()
    G = I.gaussian(256, 512, seed_cfg=0, dtype=torch.float32)
    hp = hm.HParams(K=5, eps=1e-7)
    U = run_phi(G, T, hp)
    PU.check_phi(U, G, T, hp, PU.TOL_FP32, out_is_bf16=False)


@pytest.mark.parametrize("H,W,T", [(100, 150, 32), (70, 200, 64), (130, 129, 128), (33, 47, 16)])
def test_fp32_ragged_phi(H, W, T):
    _need_gpu()
    G = I.gaussian(H, W, seed_cfg=10, layer_index=H, dtype=torch.float32)
    hp = hm.HParams(K=5, eps=1e-7)
    U = run_phi(G, T, hp)
    PU.check_phi(U, G, T, hp, PU.TOL_FP32, out_is_bf16=False)


@pytest.mark.parametrize("K", [0, 1, 3])
def test_fp32_K_sweep(K):
    _need_gpu()
    G = I.gaussian(96, 160, seed_cfg=11, dtype=torch.float32)
    hp = hm.HParams(K=K, eps=0.0)
    U = run_phi(G, 32, hp)
    PU.check_phi(U, G, 32, hp, PU.TOL_FP32, out_is_bf16=False)


@pytest.mark.parametrize("nesterov", [True, False])
def test_fp32_step_small(nesterov):
    _need_gpu()
    shapes = [(100, 150), (64, 64), (40, 300)]
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=nesterov, lr=0.02, wd=0.01, scale_c=0.2)
    Ws = [I.gaussian(h, w, seed_cfg=12, layer_index=i, tensor_id=I.TENSOR_W, dtype=torch.float32, scale=0.02) for i, (h, w) in enumerate(shapes)]
    Gs = [I.gaussian(h, w, seed_cfg=12, layer_index=i, tensor_id=I.TENSOR_G, dtype=torch.float32) for i, (h, w) in enumerate(shapes)]
    Ms = [I.gaussian(h, w, seed_cfg=12, layer_index=i, tensor_id=I.TENSOR_M, dtype=torch.float32) for i, (h, w) in enumerate(shapes)]
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    plan = hm.Plan.from_tensors(Wd, Gd, Md, 32).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        PU.check_step(Ws[i], Gs[i], Ms[i], Wd[i].cpu(), Md[i].cpu(), 32, hp, PU.TOL_FP32, storage_bf16=False)
        assert torch.equal(Gd[i].cpu(), Gs[i]), "G must be read-only"


def test_fp32_path_on_bf16_storage():
    _need_gpu()
    G = I.row_scaled_gaussian(128, 192, seed_cfg=2, dtype=torch.bfloat16)
    hp = hm.HParams(K=5, eps=1e-7)
    U = run_phi(G, 64, hp, path=hm.HIMUON_PATH_FP32)
    # bf16 output rounding alone is ~1.1e-3 relative (SURVEY 8(c) note v): the fp32 arithmetic is
    # checked by comparing against the oracle rounded to bf16, elementwise within 1 ulp.
    ref = PU.O.phi_tiled(PU.f64(G), 64, 5, *[float(np.float32(x)) for x in hm.NS_COEFFS], float(np.float32(1e-7)))
    d = np.abs(PU.f64(U) - ref)
    assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-6)


def test_ns_tiles_fp32():
    _need_gpu()
    tiles = I.gaussian(6 * 32, 32, seed_cfg=13, dtype=torch.float32).reshape(6, 32, 32).contiguous()
    tiles[2].zero_()                                   # zero tile -> zero
    out = hm.himuon_ns_tiles(tiles.to(DEV), K=5, eps=1e-7)
    torch.cuda.synchronize()
    ref = PU.O.phi_tiles(PU.f64(tiles), 5, *[float(np.float32(x)) for x in hm.NS_COEFFS], float(np.float32(1e-7)))
    got = PU.f64(out.cpu())
    assert np.all(got[2] == 0.0)
    for n in range(6):
        if n == 2:
            continue
        e = np.linalg.norm(got[n] - ref[n]) / np.linalg.norm(ref[n])
        assert e <= PU.TOL_FP32


# ----------------------------------------------------------------------------- tensor-core path, T = 128

def _tc_inputs(H, W, seed, kind="gauss"):
    if kind == "gauss":
        return I.row_scaled_gaussian(H, W, seed_cfg=seed, dtype=torch.bfloat16)
    return I.lowrank_plus_noise(H, W, 16, seed_cfg=seed, layer_index=0, tensor_id=I.TENSOR_G, dtype=torch.bfloat16)


def test_tc128_K0_normalise():
    """K = 0 returns X0 = tile / (||tile||_F + eps): exercises TMA load/store, swizzle, TMEM st/ld."""
    _need_gpu()
    G = _tc_inputs(256, 384, 20)
    hp = hm.HParams(K=0, eps=1e-7)
    U = run_phi(G, 128, hp)
    ref = PU.O.phi_tiled(PU.f64(G), 128, 0, eps=float(np.float32(1e-7)))
    d = np.abs(PU.f64(U) - ref)
    assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-12), f"max rel {np.max(d / (np.abs(ref) + 1e-30)):.3e}"


@pytest.mark.parametrize("stage", [1, 2])
def test_tc128_debug_stages(stage):
    """Intermediate accumulators of the first NS step: stage 1 = sqrt(c) X0 X0^T, stage 2 = offdiag(B)."""
    _need_gpu()
    G = _tc_inputs(128, 256, 21)
    hp = hm.HParams(K=1, eps=1e-7)
    from paper_2606_27216_b200.build import build_debug
    with B.use_library(build_debug()):        # the accumulator-dump stages exist only in the debug build
        B.debug_set_stage("tc128", stage)
        try:
            U = run_phi(G, 128, hp)
        finally:
            B.debug_set_stage("tc128", 0)
    g = PU.f64(G)
    got = PU.f64(U)
    a, b, c = [float(np.float32(x)) for x in hm.NS_COEFFS]
    for ci in range(2):
        t = g[:, 128 * ci:128 * (ci + 1)]
        X0 = t / (np.linalg.norm(t) + 1e-7)
        A = X0 @ X0.T
        blk = got[:, 128 * ci:128 * (ci + 1)].copy()
        if stage == 1:
            want = np.sqrt(c) * A                    # the kernel iterates on c^(1/4) X (see kernels_tc128.cu)
        else:
            want = b * A + c * A @ A                 # off-diagonal only: the diagonal acts as an fp32 row scaling
            np.fill_diagonal(want, 0.0)
            np.fill_diagonal(blk, 0.0)
        e = np.linalg.norm(blk - want) / np.linalg.norm(want)
        assert e <= 1e-2, f"stage {stage} tile {ci}: rel err {e:.3e}"


@pytest.mark.parametrize("K", [1, 2, 5])
@pytest.mark.parametrize("kind", ["gauss", "lowrank"])
def test_tc128_phi(K, kind):
    _need_gpu()
    G = _tc_inputs(384, 512, 22, kind)
    hp = hm.HParams(K=K, eps=1e-7)
    U = run_phi(G, 128, hp)
    PU.check_phi(U, G, 128, hp, PU.TOL_TC, out_is_bf16=True)


@pytest.mark.parametrize("H,W", [(200, 300), (128, 64), (129, 257), (1600 // 4, 192)])
def test_tc128_ragged_phi(H, W):
    """Edge tiles: zero padding on load, crop on store; gutter untouched."""
    _need_gpu()
    ld = ((W + 7) // 8) * 8 + 16
    Gfull = torch.zeros(H, ld, dtype=torch.bfloat16)
    Gfull[:, :W] = _tc_inputs(H, W, 23)
    Gd = Gfull.to(DEV)
    Ud = torch.full((H + 3, ld), 7.0, dtype=torch.bfloat16, device=DEV)      # canaries: gutter + rows past H
    hp = hm.HParams(K=5, eps=1e-7)
    plan = hm.Plan.from_tensors([Ud[:H, :W]], [Gd[:, :W]], None, 128).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    U = Ud.cpu()
    assert torch.all(U[:H, W:] == 7.0) and torch.all(U[H:] == 7.0), "wrote outside H x W"
    PU.check_phi(U[:H, :W], Gfull[:, :W], 128, hp, PU.TOL_TC, out_is_bf16=True)


def _param_set(shapes, seed, rank=16):
    Ws, Gs, Ms = [], [], []
    for i, (h, w) in enumerate(shapes):
        Gs.append(I.lowrank_plus_noise(h, w, rank, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_G))
        Ms.append(I.lowrank_plus_noise(h, w, rank, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_M))
        Ws.append(I.gaussian(h, w, seed_cfg=seed, layer_index=i, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02))
    return Ws, Gs, Ms


@pytest.mark.parametrize("nesterov,wd", [(True, 0.01), (False, 0.0)])
def test_tc128_step(nesterov, wd):
    _need_gpu()
    shapes = [(256, 256), (128, 384), (200, 136), (384, 128)]
    Ws, Gs, Ms = _param_set(shapes, 24)
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=nesterov, lr=0.02, wd=wd, scale_c=0.2)
    Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
    plan = hm.Plan.from_tensors(Wd, Gd, Md, 128).bind()
    assert plan.n_chunks == 1 and plan.n_buckets == 1
    plan.step(hp)
    torch.cuda.synchronize()
    for i in range(len(shapes)):
        PU.check_step(Ws[i], Gs[i], Ms[i], Wd[i].cpu(), Md[i].cpu(), 128, hp, PU.TOL_TC, storage_bf16=True)
        assert torch.equal(Gd[i].cpu(), Gs[i])


@pytest.mark.parametrize("T", [128, 16, 32, 64, 256])
def test_chunked_equals_unchunked(T):
    """Memory-bounded chunking is mathematically equivalent: >= 3 chunks, bit-identical,
    for every bf16 kernel path (T = 64 pairs tiles across chunk boundaries differently: still bit-identical)."""
    _need_gpu()
    shapes = [(2 * T, 3 * T), (3 * T, 2 * T), (T, T + T // 2)]
    Ws, Gs, Ms = _param_set(shapes, 25)
    hp = hm.HParams(K=5, eps=1e-7, wd=0.01)
    outs = []
    probe = hm.Plan.from_tensors(Ws, Gs, Ms, T)
    fixed = probe.workspace_bytes - 16 * probe.n_tiles
    for cap in (0, fixed + 16 * 5):
        Wd, Gd, Md = [w.to(DEV) for w in Ws], [g.to(DEV) for g in Gs], [m.to(DEV) for m in Ms]
        plan = hm.Plan.from_tensors(Wd, Gd, Md, T, workspace_cap_bytes=cap).bind()
        if cap:
            assert plan.n_chunks >= 3
        plan.step(hp)
        torch.cuda.synchronize()
        outs.append(([w.cpu() for w in Wd], [m.cpu() for m in Md]))
    for i in range(len(shapes)):
        assert torch.equal(outs[0][0][i], outs[1][0][i]) and torch.equal(outs[0][1][i], outs[1][1][i])


@pytest.mark.parametrize("path,T,dtype", [(hm.HIMUON_PATH_AUTO, 128, torch.bfloat16), (hm.HIMUON_PATH_FP32, 32, torch.float32),
                                          (hm.HIMUON_PATH_AUTO, 16, torch.bfloat16), (hm.HIMUON_PATH_AUTO, 32, torch.bfloat16),
                                          (hm.HIMUON_PATH_AUTO, 64, torch.bfloat16), (hm.HIMUON_PATH_AUTO, 256, torch.bfloat16)])
def test_indexing_bit_exact(path, T, dtype):
    """Tile indexing / reassembly with integer-tagged inputs, bit-exact (BASELINE north_star):
    lr = 0 leaves W bitwise unchanged; beta = 0 makes M' == G bitwise; gutters untouched."""
    _need_gpu()
    shapes = [(2 * T + T // 2, 3 * T), (T, T + 8), (3 * T, T // 2)]
    Ws, Gs, Ms, Wd, Gd, Md = [], [], [], [], [], []
    for i, (h, w) in enumerate(shapes):
        ld = w + 8
        for lst, dl, off in ((Ws, Wd, 0), (Gs, Gd, 1), (Ms, Md, 2)):
            full = torch.full((h, ld), -3.0, dtype=dtype)
            full[:, :w] = I.integer_tags(h, w, layer_index=3 * i + off, dtype=dtype)
            lst.append(full)
            dl.append(full.to(DEV))
    hp = hm.HParams(K=2, eps=1e-7, beta=0.0, nesterov=False, lr=0.0, wd=0.0)
    plan = hm.Plan.from_tensors([w[:, :s[1]] for w, s in zip(Wd, shapes)], [g[:, :s[1]] for g, s in zip(Gd, shapes)],
                                [m[:, :s[1]] for m, s in zip(Md, shapes)], T, path=path).bind()
    plan.step(hp)
    torch.cuda.synchronize()
    for i, (h, w) in enumerate(shapes):
        assert torch.equal(Wd[i].cpu(), Ws[i]), "lr = 0 must leave W (and its gutter) bitwise unchanged"
        assert torch.equal(Md[i].cpu()[:, :w], Gs[i][:, :w]), "beta = 0 must give M' == G bitwise"
        assert torch.all(Md[i].cpu()[:, w:] == -3.0)
        assert torch.equal(Gd[i].cpu(), Gs[i])


def test_tc128_one_hot_positions():
    """Phi with K = 0 on tiles holding a single non-zero: output non-zero exactly there (= v/(v+eps))."""
    _need_gpu()
    H, W, T = 300, 520, 128
    G = torch.zeros(H, W, dtype=torch.bfloat16)
    pos = []
    for r in range((H + T - 1) // T):
        for c in range((W + T - 1) // T):
            i = min(r * T + (37 * r + 11 * c) % T, H - 1)
            j = min(c * T + (53 * c + 29 * r) % T, W - 1)
            G[i, j] = 2.0 + r + c
            pos.append((i, j))
    U = run_phi(G, T, hm.HParams(K=0, eps=0.0))
    want = torch.zeros_like(G)
    for (i, j) in pos:
        want[i, j] = 1.0
    assert torch.equal(U, want)
