"""himuon_ns_tiles_static (include/himuon.h): the packed-tiles entry point that allocates nothing - its device scratch
is a static array inside the library - against the existing himuon_ns_tiles (caller workspace) on the same bits, on two
calls in a row that share the scratch.  Collected last on purpose (file name): the suite runs with pytest -x.
Tolerance: the per-tile relative Frobenius bar of the bf16 tensor-core path (parity_util.TOL_TC) against the existing
path's output AND against the float64 oracle; the two paths run the same deterministic kernels, so their outputs are
also required to be bitwise equal."""
import numpy as np
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm
import parity_util as PU
from paper_2606_27216_b200 import binding as B

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def _tiles(n, T, seed):
    return torch.stack([I.row_scaled_gaussian(T, T, seed_cfg=seed + i, dtype=torch.bfloat16) for i in range(n)]).to(DEV)


def _rel(a, b):
    a, b = PU.f64(a.cpu()), PU.f64(b.cpu())
    return [float(np.linalg.norm(a[i] - b[i]) / max(np.linalg.norm(b[i]), 1e-30)) for i in range(a.shape[0])]


def _check_against_existing_and_oracle(x, out_static, n_oracle):
    ref = hm.himuon_ns_tiles(x, K=5, eps=1e-7)                      # existing path, caller workspace
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out_static.float()).all())
    assert max(_rel(out_static, ref)) <= PU.TOL_TC
    assert torch.equal(out_static, ref)                             # same kernels, same bits
    ohp = PU.oracle_hp(hm.HParams(K=5, eps=1e-7))
    for i in range(n_oracle):
        o = PU.O.phi(PU.f64(x[i].cpu()), ohp.K, ohp.a, ohp.b, ohp.c, ohp.eps)
        e = np.linalg.norm(PU.f64(out_static[i].cpu()) - o) / np.linalg.norm(o)
        assert e <= PU.TOL_TC, f"tile {i}: {e:.3e}"


def test_static_scratch_entry_point_two_calls_in_a_row():
    _need_gpu()
    T = 512                                                          # the large-tile path: the kernels that use scratch
    nmax = hm.himuon_ns_tiles_static_max_tiles(T)
    assert nmax == 12
    xa, xb = _tiles(nmax, T, 910), _tiles(5, T, 940)                 # a full scratch, then a smaller batch over its remains
    xs = _tiles(37, 128, 970)                                        # a fused-kernel tile size: only the table area is used
    oa = torch.full_like(xa, float("nan"))
    ob = torch.full_like(xb, float("nan"))
    os_ = torch.full_like(xs, float("nan"))
    os2 = torch.full_like(xs, float("nan"))
    torch.cuda.synchronize()
    hm.himuon_ns_tiles_static(xa, oa, K=5, eps=1e-7)                 # call 1 (first use also loads the kernels' code)
    hm.himuon_ns_tiles_static(xs, os_, K=5, eps=1e-7)                # call 2, straight after: rewrites the table area
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    hm.himuon_ns_tiles_static(xb, ob, K=5, eps=1e-7)                 # call 3, same stream, over the remains of call 1
    hm.himuon_ns_tiles_static(xs, os2, K=5, eps=1e-7)                # call 4
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                     # no device memory taken once the code is loaded
    assert torch.equal(os2, os_)
    _check_against_existing_and_oracle(xa, oa, 2)
    _check_against_existing_and_oracle(xb, ob, 1)
    _check_against_existing_and_oracle(xs, os_, 2)
    # call 1's input once more, over the scratch the other calls left: identical bits
    oa2 = torch.full_like(xa, float("nan"))
    hm.himuon_ns_tiles_static(xa, oa2, K=5, eps=1e-7)
    torch.cuda.synchronize()
    assert torch.equal(oa2, oa)


def test_static_scratch_entry_point_rejects_what_does_not_fit():
    _need_gpu()
    T = 512
    n = hm.himuon_ns_tiles_static_max_tiles(T) + 1
    x = torch.zeros(n, T, T, dtype=torch.bfloat16, device=DEV)
    out = torch.full_like(x, 7.0)
    with pytest.raises(hm.HimuonError) as ei:
        hm.himuon_ns_tiles_static(x, out, K=5, eps=1e-7)
    assert ei.value.status == B.HIMUON_ERR_WORKSPACE_TOO_SMALL
    assert "at most 12" in str(ei.value) and "HIMUON_STATIC_SCRATCH_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                  # nothing was enqueued
    assert hm.himuon_ns_tiles_static_max_tiles(48) == 0              # not a tile size
    with pytest.raises(ValueError):
        hm.himuon_ns_tiles_static(x.float(), out.float())            # bf16 only
