"""One tiny ragged Algorithm-4.1 step per kernel of the library, each checked against the float64 oracle.

Small enough to run under `compute-sanitizer` (racecheck / synccheck / memcheck): the
hand-written mbarrier / TMEM / TMA pipelines are exactly the kind of code those tools exist for.  The command

    compute-sanitizer --tool <tool> python -m pytest tests/test_gpu_tiny_all_kernels.py -m gpu -q

is refused by this GPU pool (profiles/r2_sanitizer.md says what was asked and what stands in for it).
"""
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm
import parity_util as PU

pytestmark = pytest.mark.gpu
DEV = "cuda"

CASES = [
    # id, storage dtype, path, T, (H, W), tolerance
    ("warp16", torch.bfloat16, hm.HIMUON_PATH_AUTO, 16, (40, 50), PU.TOL_TC),
    ("warp32", torch.bfloat16, hm.HIMUON_PATH_AUTO, 32, (70, 96), PU.TOL_TC),
    ("tc64", torch.bfloat16, hm.HIMUON_PATH_AUTO, 64, (200, 136), PU.TOL_TC),
    ("tc128", torch.bfloat16, hm.HIMUON_PATH_AUTO, 128, (200, 328), PU.TOL_TC),
    ("tc256", torch.bfloat16, hm.HIMUON_PATH_AUTO, 256, (300, 640), PU.TOL_TC),
    ("tc128_fp8", torch.bfloat16, hm.HIMUON_PATH_FP8, 128, (200, 328), 0.15),
    ("tc256_fp8", torch.bfloat16, hm.HIMUON_PATH_FP8, 256, (300, 640), 0.15),
    ("simt_fp32", torch.float32, hm.HIMUON_PATH_AUTO, 64, (100, 130), PU.TOL_FP32),
    ("simt_bf16", torch.bfloat16, hm.HIMUON_PATH_FP32, 32, (70, 96), 5e-3),
    ("large512", torch.bfloat16, hm.HIMUON_PATH_AUTO, 512, (600, 1032), PU.TOL_TC),
]


@pytest.mark.parametrize("name,dtype,path,T,shape,tol", CASES, ids=[c[0] for c in CASES])
def test_tiny_ragged_step(name, dtype, path, T, shape, tol):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    H, W = shape
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    G = I.lowrank_plus_noise(H, W, 8, seed_cfg=41, layer_index=0, tensor_id=I.TENSOR_G, dtype=dtype)
    M0 = I.lowrank_plus_noise(H, W, 8, seed_cfg=41, layer_index=0, tensor_id=I.TENSOR_M, dtype=dtype)
    W0 = I.gaussian(H, W, seed_cfg=41, layer_index=0, tensor_id=I.TENSOR_W, dtype=dtype, scale=0.02)
    Wd, Gd, Md = W0.to(DEV), G.to(DEV), M0.to(DEV)
    plan = hm.Plan.from_tensors([Wd], [Gd], [Md], T, path=path).bind()
    plan.step(hp)
    plan.step(hp)          # a second step reuses every buffer, barrier phase and prefetch of the persistent kernels
    torch.cuda.synchronize()
    plan.destroy()
    bf = dtype == torch.bfloat16
    # second step from the GPU's own stored state of the first (the stored M', W' are what it reads back)
    plan1 = hm.Plan.from_tensors([W0.to(DEV)], [Gd], [M0.to(DEV)], T, path=path).bind()
    plan1.step(hp)
    torch.cuda.synchronize()
    Wmid, Mmid = plan1._keep[0][0].cpu(), plan1._keep[2][0].cpu()
    plan1.destroy()
    PU.check_step(W0, G, M0, Wmid, Mmid, T, hp, tol, storage_bf16=bf)
    PU.check_step(Wmid, G, Mmid, Wd.cpu(), Md.cpu(), T, hp, tol, storage_bf16=bf)
