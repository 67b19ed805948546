"""GPU tests of the fp8 (e4m3) variants of the T = 128 and T = 256 kernels (HIMUON_PATH_FP8; the F8 template
variants in csrc/kernels_tc128.cu and csrc/kernels_tc256.cu; SURVEY 8(f3);
PAPER.md:410-424 section 6.5, :440).  Only the operands of the three products of a Newton-Schulz step are e4m3;
everything else is the bf16 kernel's fp32 arithmetic.  Tolerance: per-tile relative Frobenius error <= 0.15 against
the float64 oracle (0.07-0.12 measured in emulation on these recipes; the paper reports an
operator gap of 0.059 for its own T = 128 fp8 update)."""
import numpy as np
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm
from paper_2606_27216_b200 import binding as B
import parity_util as PU

pytestmark = pytest.mark.gpu
DEV = "cuda"
TOL_FP8 = 0.15
SX, SO, SB = 256.0, 128.0, 128.0          # the kernel's operand scales (its header)


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def _e4m3(x):
    """Round float64 values to e4m3 (torch's conversion: round to nearest even, subnormals) and back."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float32)).clamp(-448, 448)
    return t.to(torch.float8_e4m3fn).to(torch.float64).numpy()


def _inputs(H, W, seed, kind="gauss"):
    if kind == "gauss":
        return I.row_scaled_gaussian(H, W, seed_cfg=seed, dtype=torch.bfloat16)
    return I.lowrank_plus_noise(H, W, 16, seed_cfg=seed, layer_index=0, tensor_id=I.TENSOR_G, dtype=torch.bfloat16)


def _run_phi(G, hp, T=128):
    Gd = G.to(DEV)
    Ud = torch.full_like(Gd, float("nan"))
    plan = hm.Plan.from_tensors([Ud], [Gd], None, T, path=hm.HIMUON_PATH_FP8).bind()
    plan.phi(hp)
    torch.cuda.synchronize()
    plan.destroy()
    return Ud.cpu()


def test_fp8_K0_normalise():
    """K = 0 touches no product: X0 = tile / (||tile||_F + eps) to one bf16 rounding."""
    _need_gpu()
    G = _inputs(256, 384, 20)
    U = _run_phi(G, hm.HParams(K=0, eps=1e-7))
    ref = PU.O.phi_tiled(PU.f64(G), 128, 0, eps=float(np.float32(1e-7)))
    d = np.abs(PU.f64(U) - ref)
    assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-12)


@pytest.mark.parametrize("stage", [1, 2])
def test_fp8_debug_stages(stage):
    """Accumulators of the first NS step, raw (scaled): stage 1 = (s_X Xq)(s_X Xq)^T with Xq the e4m3 operand,
    stage 2 off-diagonal = s_O^2 (beta Ah + Ah^2).  Checks the e4m3 operand layouts in shared and tensor memory,
    the K-major / MN-major descriptors and the kind::f8f6f4 instruction descriptor."""
    _need_gpu()
    G = _inputs(128, 256, 21)
    from paper_2606_27216_b200.build import build_debug
    with B.use_library(build_debug()):        # the accumulator-dump stages exist only in the debug build
        B.debug_set_stage("tc128_fp8", stage)
        try:
            U = _run_phi(G, hm.HParams(K=1, eps=1e-7))
        finally:
            B.debug_set_stage("tc128_fp8", 0)
    g, got = PU.f64(G), PU.f64(U)
    a, b, c = [float(np.float32(x)) for x in hm.NS_COEFFS]
    for ci in range(2):
        t = g[:, 128 * ci:128 * (ci + 1)]
        Xh = c ** 0.25 * t / (np.linalg.norm(t) + 1e-7)          # the kernel iterates on c^(1/4) X
        blk = got[:, 128 * ci:128 * (ci + 1)].copy()
        if stage == 1:
            Xq = _e4m3(SX * Xh)
            want = Xq @ Xq.T
            tol = 1e-2                                            # fp32 accumulation + one bf16 rounding on output
        else:
            Ah = Xh @ Xh.T
            want = SO * SO * ((b / np.sqrt(c)) * Ah + Ah @ Ah)
            np.fill_diagonal(want, 0.0)
            np.fill_diagonal(blk, 0.0)
            tol = 0.1                                             # two e4m3 operand roundings
        e = np.linalg.norm(blk - want) / np.linalg.norm(want)
        assert e <= tol, f"stage {stage} tile {ci}: rel err {e:.3e}"


@pytest.mark.parametrize("T", [128, 256])
@pytest.mark.parametrize("K", [1, 5])
@pytest.mark.parametrize("kind", ["gauss", "lowrank"])
def test_fp8_phi(K, kind, T):
    _need_gpu()
    G = _inputs(3 * T, 4 * T, 22, kind)
    hp = hm.HParams(K=K, eps=1e-7)
    U = _run_phi(G, hp, T)
    worst = PU.check_phi(U, G, T, hp, TOL_FP8, out_is_bf16=True)
    print(f"FP8 phi T={T} K={K} {kind}: worst per-tile error {worst:.3e}")


def test_fp8_K0_normalise_T256():
    _need_gpu()
    G = _inputs(512, 768, 20)
    U = _run_phi(G, hm.HParams(K=0, eps=1e-7), 256)
    ref = PU.O.phi_tiled(PU.f64(G), 256, 0, eps=float(np.float32(1e-7)))
    d = np.abs(PU.f64(U) - ref)
    assert np.all(d <= PU.BF16_ULP * np.abs(ref) + 1e-12)


@pytest.mark.parametrize("T,H,W", [(128, 200, 328), (256, 300, 640), (256, 300, 520)])
def test_fp8_ragged_step(T, H, W):
    """Full step with edge tiles (zero padding on load, crop on store) on the fp8 path, one tolerance for all.
    The last case has a 44 x 8 corner block: with so few singular directions e4m3 rounding errors do not average
    out (0.19 measured when the e4m3 kernel ran it), so the plan routes edge tiles with fewer than 32 live rows or
    columns to the bf16 kernel of the same tile size (its own bucket) - checked here through the work list."""
    _need_gpu()
    tol = TOL_FP8
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    G = _inputs(H, W, 31)
    M0 = I.gaussian(H, W, seed_cfg=31, layer_index=0, tensor_id=I.TENSOR_M, dtype=torch.bfloat16)
    W0 = (0.02 * I.gaussian(H, W, seed_cfg=31, layer_index=0, tensor_id=I.TENSOR_W, dtype=torch.float32)).to(torch.bfloat16)
    Wd, Gd, Md = W0.to(DEV), G.to(DEV), M0.to(DEV)
    plan = hm.Plan.from_tensors([Wd], [Gd], [Md], T, path=hm.HIMUON_PATH_FP8).bind()
    small = [(r, c) for r in range(-(-H // T)) for c in range(-(-W // T))
             if min(T, H - r * T) < 32 or min(T, W - c * T) < 32]
    lrc, offs, cT = plan.worklist()
    assert plan.n_buckets == (2 if small else 1) and plan.n_tiles == -(-H // T) * -(-W // T)
    if small:   # the second bucket (bf16 kernel) holds exactly the small edge tiles
        assert sorted((int(r), int(c)) for _, r, c in lrc[offs[1]:]) == sorted(small)
    plan.step(hp)
    torch.cuda.synchronize()
    plan.destroy()
    PU.check_step(W0, G, M0, Wd.cpu(), Md.cpu(), T, hp, tol, storage_bf16=True)


def test_fp8_path_serves_T128_and_T256_only():
    _need_gpu()
    G = _inputs(512, 512, 40).to(DEV)
    U = torch.empty_like(G)
    for T in (64, 512):
        with pytest.raises(hm.HimuonError):
            hm.Plan.from_tensors([U], [G], None, T, path=hm.HIMUON_PATH_FP8)
    Gf = G.float()
    with pytest.raises(hm.HimuonError):
        hm.Plan.from_tensors([torch.empty_like(Gf)], [Gf], None, 128, path=hm.HIMUON_PATH_FP8)


@pytest.mark.parametrize("T", [128, 256])
def test_fp8_capacity_diagnostic(T):
    """Table 3's fp8e4m3 column: recovered items with e4m3 inner products agree with the fp64 count
    to well within the seed standard deviation (the paper: 406.8 against 408.0 at T = 128, 485.8 against 486.4 at
    T = 256, sigma 13-15)."""
    _need_gpu()
    prob = I.assoc_memory_problem(1024, 4096, 1.5, 10240, seed=0)
    ref = PU.O.phi_tiled(prob.G0, T, K=5, eps=1e-7)
    n_ref = I.recovered_items(prob, -ref)
    ref_b = PU.O.phi_tiled(I.bf16_round_f64(prob.G0), T, K=5, eps=1e-7)
    G = torch.from_numpy(prob.G0).to(torch.bfloat16)
    got = PU.f64(_run_phi(G, hm.HParams(K=5, eps=1e-7), T))
    n_got = I.recovered_items(prob, -got)
    gap = float(np.linalg.norm(got - ref) / np.linalg.norm(ref))
    gap_b = float(np.linalg.norm(got - ref_b) / np.linalg.norm(ref_b))
    print(f"CAPACITY fp8 T={T}: recovered {n_got} (fp64 oracle {n_ref}), operator gap {gap:.3e}, "
          f"to the same-input oracle {gap_b:.3e}")
    assert abs(n_got - n_ref) <= 15
    assert gap_b <= TOL_FP8


@pytest.mark.parametrize("T,N", [(128, 37), (256, 9)])
def test_fp8_ns_tiles_packed_batch(T, N):
    """himuon_ns_tiles on a packed [N, T, T] batch (the Fig. 7 workload) through the fp8 path."""
    _need_gpu()
    tiles = I.row_scaled_gaussian(N * T, T, seed_cfg=50, dtype=torch.bfloat16).reshape(N, T, T).contiguous()
    out = hm.himuon_ns_tiles(tiles.to(DEV), K=5, eps=1e-7, path=hm.HIMUON_PATH_FP8)
    torch.cuda.synchronize()
    got = PU.f64(out.cpu())
    worst = 0.0
    for i in range(N):
        ref = PU.O.phi(PU.f64(tiles[i]), 5, eps=float(np.float32(1e-7)))
        worst = max(worst, float(np.linalg.norm(got[i] - ref) / np.linalg.norm(ref)))
    assert np.all(np.isfinite(got)) and worst <= TOL_FP8, f"worst tile error {worst:.3e}"


@pytest.mark.parametrize("T", [128, 256])
def test_fp8_chunked_equals_unchunked(T):
    """The workspace cap splits the work list into chunks; chunking must not change a bit."""
    _need_gpu()
    G = _inputs(4 * T, 6 * T, 51)
    hp = hm.HParams(K=5, eps=1e-7)
    probe = hm.Plan.from_tensors([torch.empty_like(G)], [G], None, T, path=hm.HIMUON_PATH_FP8)
    fixed = probe.workspace_bytes - 16 * probe.n_tiles
    outs = []
    for cap in (0, fixed + 16 * 5):
        Gd = G.to(DEV)
        Ud = torch.full_like(Gd, float("nan"))
        plan = hm.Plan.from_tensors([Ud], [Gd], None, T, path=hm.HIMUON_PATH_FP8, workspace_cap_bytes=cap).bind()
        plan.phi(hp)
        torch.cuda.synchronize()
        outs.append((Ud.cpu(), plan.n_chunks))
        plan.destroy()
    assert outs[0][1] == 1 and outs[1][1] >= 3
    assert torch.equal(outs[0][0], outs[1][0])
