"""CPU-only tests of the C-ABI library's host logic: it loads, exports every symbol declared in
include/himuon.h, validates arguments, and its planner (work list, buckets, memory-bounded
chunking) agrees with the oracle's enumeration and with the numbers the paper prints."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import himuon_inputs as I
import paper_2606_27216_b200 as hm
from paper_2606_27216_b200 import binding as B
from paper_2606_27216_b200.build import build
from oracle import himuon_oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    build()


def _layers(shapes, dtype=hm.HIMUON_BF16, Ts=None):
    return [hm.himuon_layer(hm.shape_mat(h, w, dtype), hm.shape_mat(h, w, dtype), hm.shape_mat(h, w, dtype),
                            0 if Ts is None else Ts[i]) for i, (h, w) in enumerate(shapes)]


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "himuon.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(himuon_[a-z0-9_]+)\s*\(", hdr))
    assert {"himuon_plan_create", "himuon_step", "himuon_phi", "himuon_ns_tiles", "himuon_plan_bind"} <= names
    lib = C.CDLL(B.LIB_PATH)
    for n in sorted(names):
        assert hasattr(lib, n), f"libhimuon.so does not export {n}"


def test_status_strings():
    lib = B._lib()
    assert lib.himuon_status_string(0) == b"HIMUON_OK"
    assert lib.himuon_status_string(2) == b"HIMUON_ERR_UNSUPPORTED"


@pytest.mark.parametrize("shapes,T", [([(256, 512)], 64), ([(1600, 1600), (1600, 6400), (6400, 1600)], 128),
                                      ([(100, 90), (33, 700)], 32), ([(5, 3)], 16)])
def test_worklist_matches_oracle_enumeration(shapes, T):
    """R = ceil(H/T), C = ceil(W/T); layer order then r-major."""
    p = hm.Plan(_layers(shapes), T)
    lrc, offs, cT = p.worklist()
    want = O.enumerate_tiles(shapes, [T] * len(shapes))
    assert [tuple(x) for x in lrc.tolist()] == want
    assert p.n_tiles == len(want) and p.n_buckets == 1 and p.n_chunks == 1
    assert offs.tolist() == [0, len(want)]


def test_config1_tile_count_reading_Q1():
    # 256x512 at T=64 is 4 x 8 = 32 tiles by PAPER.md:48-49 (BASELINE's "8 tiles" is T=128)
    assert hm.Plan(_layers([(256, 512)], hm.HIMUON_F32), 64).n_tiles == 32
    assert hm.Plan(_layers([(256, 512)], hm.HIMUON_F32), 128).n_tiles == 8


def test_tile_counts_of_the_benchmark_configs():
    # SURVEY.md 8(a) [derived]: config 2 = 5184, config 4 = 94848, config 5 = 425984 tiles at T=128
    for spec, n in ((I.gpt2_small_spec(), 5184), (I.gpt2_xl_spec(), 94848), (I.llama3_8b_spec(), 425984)):
        p = hm.Plan(_layers([(l.H, l.W) for l in spec.layers]), 128)
        assert p.n_tiles == n
        assert p.n_chunks == 1


def test_paper_planner_numbers(paper_numbers):
    """1680 tiles -> 1 call; 5376 tiles -> two chunks of 2688 (T=512)."""
    T = int(paper_numbers["tile_size"])
    blocks = int(paper_numbers["qwen3_blocks"])

    def n_tiles(key):
        shapes = [tuple(int(x) for x in s.split("x")) for s in paper_numbers[key].split()]
        return blocks * sum(-(-h // T) * -(-w // T) for h, w in shapes)

    n06, n17 = n_tiles("shapes_0p6b"), n_tiles("shapes_1p7b")
    assert n06 == int(paper_numbers["tiles_0p6b"]) and n17 == int(paper_numbers["tiles_1p7b"])
    per_tile = 3 * T * T * 2                      # paper's staged model: in + intermediate + out, bf16
    for cap_tiles in (2688, 3000, 5375):          # any budget admitting 2688..5375 tiles
        offs = hm.himuon_plan_chunks(n17, per_tile, 0, cap_tiles * per_tile)
        assert offs == [0, int(paper_numbers["chunk_size_1p7b"]), n17]
        assert hm.himuon_plan_chunks(n06, per_tile, 0, cap_tiles * per_tile) == [0, n06]


@pytest.mark.parametrize("n,per,fixed,cap", [(10, 7, 3, 30), (1000, 16, 1000, 5000), (7, 1, 0, 2), (5, 0, 0, 1), (0, 4, 0, 100)])
def test_chunk_rule_matches_oracle(n, per, fixed, cap):
    assert hm.himuon_plan_chunks(n, per, fixed, cap) == O.chunk_offsets(n, per, cap, fixed)


def test_chunk_rule_too_small():
    with pytest.raises(hm.HimuonError) as e:
        hm.himuon_plan_chunks(10, 100, 0, 50)
    assert e.value.status == B.HIMUON_ERR_WORKSPACE_TOO_SMALL


def test_chunked_plan_is_balanced_and_fewest():
    shapes = [(1600, 1600)] * 3
    full = hm.Plan(_layers(shapes), 128)
    fixed = full.workspace_bytes - full.n_tiles * 16
    p = hm.Plan(_layers(shapes), 128, workspace_cap_bytes=fixed + 16 * 100)
    lrc, offs, _ = p.worklist()
    sizes = np.diff(offs)
    assert p.n_chunks == -(-full.n_tiles // 100) and sizes.max() - sizes.min() <= 1 and sizes.max() <= 100
    assert p.workspace_bytes <= fixed + 16 * 100
    assert [tuple(x) for x in lrc.tolist()] == O.enumerate_tiles(shapes, [128] * 3)   # order unchanged


def test_runtime_tile_schedule_buckets():
    """Reading Q13: per-layer T; tiles bucketed by (T, dtype, path); momentum is not
    part of the plan, so re-planning cannot touch it."""
    shapes = [(256, 256), (128, 512), (256, 256), (512, 128)]
    Ts = [128, 64, 128, 32]
    p = hm.Plan(_layers(shapes, Ts=Ts), 128)
    lrc, offs, cT = p.worklist()
    assert p.n_buckets == 3 and cT.tolist() == [128, 64, 32]
    want = []
    for T in (128, 64, 32):
        want += [x for x in O.enumerate_tiles(shapes, Ts) if Ts[x[0]] == T]
    assert [tuple(x) for x in lrc.tolist()] == want


def test_full_branch_is_one_padded_tile():
    # T >= max(H,W): R = C = 1; run as the smallest supported tile >= max(H,W)
    p = hm.Plan(_layers([(100, 90)]), 128)
    lrc, _, cT = p.worklist()
    assert lrc.tolist() == [[0, 0, 0]] and cT.tolist() == [128]
    p = hm.Plan(_layers([(20, 30)], hm.HIMUON_F32), 128)
    assert p.worklist()[2].tolist() == [32]
    # larger than every tile kernel: one whole-matrix item on the large-tile (cuBLAS) path
    p = hm.Plan(_layers([(4096, 4096)]), 8192)
    assert p.n_tiles == 1 and p.workspace_bytes > 2 * 4096 * 4096 * 4


def test_argument_validation():
    S = B.HIMUON_ERR_INVALID_ARG
    for bad in ([(0, 5)], [(5, -1)]):
        with pytest.raises(hm.HimuonError) as e:
            hm.Plan(_layers(bad), 32)
        assert e.value.status == S
    with pytest.raises(hm.HimuonError) as e:      # ld < W
        hm.Plan([hm.himuon_layer(hm.shape_mat(8, 8, ld=4), hm.shape_mat(8, 8), hm.shape_mat(8, 8), 0)], 16)
    assert e.value.status == S
    with pytest.raises(hm.HimuonError) as e:      # T not a supported size
        hm.Plan(_layers([(256, 256)]), 48)
    assert e.value.status == S
    with pytest.raises(hm.HimuonError) as e:      # bad dtype
        hm.Plan(_layers([(256, 256)], dtype=7), 32)
    assert e.value.status == S
    p = hm.Plan(_layers([(256, 256)]), 128)       # unbound / unbindable plan
    with pytest.raises(hm.HimuonError) as e:
        p.step(hm.HParams())
    assert e.value.status == B.HIMUON_ERR_NOT_BOUND
    lib = B._lib()
    assert lib.himuon_plan_bind(p._h, None, 0, None) == S
    assert lib.himuon_ns_tiles(None, None, -1, 32, 0, 0, 5, 1.0, 1.0, 1.0, 0.0, None, 0, None) == S
    assert lib.himuon_ns_tiles(None, None, 4, 48, 0, 0, 5, 1.0, 1.0, 1.0, 0.0, None, 0, None) == S
    assert lib.himuon_ns_tiles(None, None, 0, 32, 0, 0, 5, 1.0, 1.0, 1.0, 0.0, None, 0, None) == B.HIMUON_OK


def test_tma_alignment_is_checked():
    # tensor-core path: ld*2 must be a multiple of 16 bytes
    with pytest.raises(hm.HimuonError) as e:
        hm.Plan([hm.himuon_layer(hm.himuon_mat(256, 256, 256, 257, 1), hm.himuon_mat(256, 256, 256, 257, 1),
                                 hm.himuon_mat(256, 256, 256, 257, 1), 0)], 128)
    assert e.value.status == B.HIMUON_ERR_UNSUPPORTED


def test_supported_tile_sizes_per_dtype_and_path():
    assert hm.himuon_supported_tile_sizes(hm.HIMUON_F32) == [16, 32, 64, 128, 256, 512]
    assert hm.himuon_supported_tile_sizes(hm.HIMUON_BF16) == [16, 32, 64, 128, 256, 512]
    assert hm.himuon_supported_tile_sizes(hm.HIMUON_BF16, hm.HIMUON_PATH_FP32) == [16, 32, 64, 128, 256, 512]
    # T = 256 without a tile kernel (fp32 storage; bf16 width not a multiple of 8) and T = 512 run on the
    # large-tile path, whose scratch is part of the plan's workspace
    small = hm.Plan(_layers([(512, 512)]), 256)
    assert small.n_tiles == 4 and small.workspace_bytes < 1 << 20
    # fp32 storage: fp32 cuBLAS products (32 MB of cuBLAS workspace inside the scratch)
    assert hm.Plan(_layers([(512, 512)], hm.HIMUON_F32), 256).workspace_bytes > 32 << 20
    # bf16: the tcgen05 large-tile path - per tile the iterate as three bf16 arrays (hi x 2, lo) and two bf16 r x r operands
    pl = hm.Plan(_layers([(512, 304), (512, 300)]), 256)
    assert pl.n_buckets == 2 and pl.workspace_bytes > 4 * 256 * 256 * (2 + 2 + 2 + 2 + 2)
    p = hm.Plan(_layers([(1024, 1536)]), 512)
    assert p.n_tiles == 6 and p.workspace_bytes > 6 * 512 * 512 * (2 + 2 + 2 + 2 + 2)
    assert hm.Plan(_layers([(200, 256)]), 256).n_tiles == 1     # full-matrix branch served by the T = 256 kernel
    with pytest.raises(hm.HimuonError) as e:                    # the scratch counts against the workspace cap
        hm.Plan(_layers([(4096, 4096)]), 8192, workspace_cap_bytes=64 << 20)
    assert e.value.status == B.HIMUON_ERR_WORKSPACE_TOO_SMALL


def test_kernel_paths_bucket_the_work_list():
    """Buckets by (T, dtype, kernel path): bf16 T = 16/32 -> warp kernel, 64/128/256 -> tcgen05
    kernels, a bf16 width that is not a multiple of 8 -> fp32 kernel; one bucket per distinct key."""
    shapes = [(256, 256), (256, 256), (256, 256), (256, 256), (256, 256), (256, 250)]
    p = hm.Plan(_layers(shapes, Ts=[16, 32, 64, 128, 256, 128]), 128)
    assert p.n_buckets == 6
    assert p.n_tiles == 256 + 64 + 16 + 4 + 1 + 4
    _, offs, cT = p.worklist()
    assert cT.tolist() == [16, 32, 64, 128, 256, 128] and p.n_chunks == 6


def test_rectangular_tiles_plan():
    """T_w != T: R = ceil(H/T), C = ceil(W/T_w), both extents powers of two in 16..2048."""
    L = [hm.himuon_layer(hm.shape_mat(300, 500), hm.shape_mat(300, 500), hm.shape_mat(300, 500), 128, 32)]
    p = hm.Plan(L, 128)
    lrc, _, cT = p.worklist()
    assert p.n_tiles == 3 * 16 and lrc[-1].tolist() == [0, 2, 15] and cT.tolist() == [128]
    L[0].T_w = 128                                   # T_w == T is the square case: tensor-core kernel, no scratch
    assert hm.Plan(L, 128).workspace_bytes < 1 << 20
    L[0].T_w = 48
    with pytest.raises(hm.HimuonError) as e:
        hm.Plan(L, 128)
    assert e.value.status == B.HIMUON_ERR_INVALID_ARG
    L[0].T, L[0].T_w = 512, 1024                     # one tile covers the matrix: full-matrix branch
    assert hm.Plan(L, 128).n_tiles == 1


def test_chunk_rule_properties():
    """Properties of the memory-bounded chunk rule (fewest chunks that fit, balanced sizes)
    over random instances, against what the rule must guarantee rather than against a second implementation."""
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=300, deadline=None)
    @given(n=st.integers(0, 200000), per=st.integers(1, 1 << 20), fixed=st.integers(0, 1 << 20), slack=st.integers(0, 1 << 24))
    def check(n, per, fixed, slack):
        cap = fixed + per + slack                       # room for at least one item
        offs = hm.himuon_plan_chunks(n, per, fixed, cap)
        assert offs[0] == 0 and offs[-1] == n and all(b > a for a, b in zip(offs, offs[1:]))
        sizes = np.diff(offs)
        if n == 0:
            assert len(offs) == 1
            return
        per_max = (cap - fixed) // per
        assert sizes.max() <= per_max                    # every chunk fits under the cap
        assert len(sizes) == -(-n // per_max)            # and there are as few chunks as that allows
        assert sizes.max() - sizes.min() <= 1            # balanced (5376 -> 2 x 2688)

    check()


def test_fp8_path_is_opt_in_and_T128_T256_only():
    """HIMUON_PATH_FP8 (e4m3 operands, include/himuon.h): bf16 storage, T = 128 or 256, width a multiple of 8 - everything
    else is refused at plan time, never silently served by another kernel; AUTO never selects it."""
    U = B.HIMUON_ERR_UNSUPPORTED
    assert hm.himuon_supported_tile_sizes(hm.HIMUON_BF16, hm.HIMUON_PATH_FP8) == [128, 256]
    assert hm.himuon_supported_tile_sizes(hm.HIMUON_F32, hm.HIMUON_PATH_FP8) == []
    p = hm.Plan(_layers([(512, 768), (100, 128)]), 128, path=hm.HIMUON_PATH_FP8)
    assert p.n_tiles == 24 + 1 and p.n_buckets == 1
    assert hm.Plan(_layers([(512, 768)]), 256, path=hm.HIMUON_PATH_FP8).n_tiles == 6
    for shapes, T, kw in (([(512, 512)], 64, {}), ([(512, 500)], 256, {}), ([(512, 512)], 512, {}),
                          ([(512, 500)], 128, {}), ([(512, 512)], 128, {"dtype": hm.HIMUON_F32})):
        with pytest.raises(hm.HimuonError) as e:
            hm.Plan(_layers(shapes, **kw), T, path=hm.HIMUON_PATH_FP8)
        assert e.value.status == U, (shapes, T, kw)
    with pytest.raises(hm.HimuonError) as e:                    # an unknown path value is an argument error
        hm.Plan(_layers([(256, 256)]), 128, path=3)
    assert e.value.status == B.HIMUON_ERR_INVALID_ARG


def test_nonpositive_c_is_refused_on_the_tensor_core_paths():
    """The bf16 / e4m3 tensor-core kernels iterate on c^(1/4) X: c <= 0 - e.g. the cubic
    iteration (1.5, -0.5, 0) - must be refused before any launch, not turned into NaN weights.  The check is pure
    argument validation, so it fires even on an unbound plan; the fp32 path takes any finite (a, b, c)."""
    lib = B._lib()
    for c, want_tc in ((0.0, B.HIMUON_ERR_UNSUPPORTED), (-1.0, B.HIMUON_ERR_UNSUPPORTED), (2.0315, B.HIMUON_ERR_NOT_BOUND)):
        hp = hm.HParams(a=1.5, b=-0.5, c=c).to_c()
        for T in (64, 128, 256, 512):
            p = hm.Plan(_layers([(512, 512)]), T)
            assert lib.himuon_step(p._h, C.byref(hp), None) == want_tc, (c, T)
            assert lib.himuon_phi(p._h, C.byref(hp), None) == want_tc, (c, T)
        p = hm.Plan(_layers([(512, 512)]), 128, path=hm.HIMUON_PATH_FP8)
        assert lib.himuon_phi(p._h, C.byref(hp), None) == want_tc
        # the warp kernel (T = 16, 32: plain state) and fp32 arithmetic (FP32 path, fp32 storage): accepted ("not bound" here)
        p = hm.Plan(_layers([(512, 512)]), 16)
        assert lib.himuon_phi(p._h, C.byref(hp), None) == B.HIMUON_ERR_NOT_BOUND
        p = hm.Plan(_layers([(512, 512)]), 64, path=hm.HIMUON_PATH_FP32)
        assert lib.himuon_phi(p._h, C.byref(hp), None) == B.HIMUON_ERR_NOT_BOUND
        p = hm.Plan(_layers([(512, 512)], hm.HIMUON_F32), 64)
        assert lib.himuon_phi(p._h, C.byref(hp), None) == B.HIMUON_ERR_NOT_BOUND
    # himuon_ns_tiles validates before touching any pointer
    for T, dt, want in ((128, hm.HIMUON_BF16, B.HIMUON_ERR_UNSUPPORTED), (64, hm.HIMUON_F32, B.HIMUON_OK)):
        st = lib.himuon_ns_tiles(None, None, 0, T, dt, hm.HIMUON_PATH_AUTO, 5, 1.5, -0.5, 0.0, 1e-7, None, 0, None)
        assert st == want, (T, dt, st)


def test_plans_from_two_threads():
    """The library keeps no unsynchronised process-global state on the planning path: two host threads building,
    inspecting and destroying plans concurrently get the same work lists as one thread."""
    import threading
    shapes = [(1600, 1600), (1600, 6400), (6400, 1600)] * 4
    want = O.enumerate_tiles(shapes, [128] * len(shapes))
    errors = []

    def worker(seed):
        try:
            for i in range(20):
                T = (64, 128, 256)[(i + seed) % 3]
                p = hm.Plan(_layers(shapes), T, workspace_cap_bytes=(1 << 20) if i % 2 else 0)
                lrc, offs, cT = p.worklist()
                if T == 128 and [tuple(x) for x in lrc.tolist()] != want:
                    errors.append("work list differs")
                if offs[-1] != p.n_tiles:
                    errors.append("chunk offsets")
                p.destroy()
        except Exception as e:        # noqa: BLE001
            errors.append(repr(e))

    ts = [threading.Thread(target=worker, args=(s,)) for s in range(2)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors


def test_fp8_plan_routes_small_edge_tiles_to_the_bf16_kernel():
    """An e4m3 layer's edge tiles with fewer than 32 live rows or columns form a second bucket (bf16 kernel, same T);
    every tile appears exactly once (buckets by kernel path)."""
    p = hm.Plan(_layers([(300, 520), (256, 512)]), 256, path=hm.HIMUON_PATH_FP8)
    lrc, offs, cT = p.worklist()
    assert p.n_buckets == 2 and p.n_chunks == 2 and cT.tolist() == [256, 256]
    all_tiles = sorted(tuple(x) for x in lrc.tolist())
    assert all_tiles == sorted(O.enumerate_tiles([(300, 520), (256, 512)], [256, 256]))
    assert sorted(tuple(x) for x in lrc[offs[1]:].tolist()) == [(0, 0, 2), (0, 1, 2)]     # 8 live columns
    # no small edge tile: one bucket
    assert hm.Plan(_layers([(300, 640)]), 256, path=hm.HIMUON_PATH_FP8).n_buckets == 1
