"""Microbenchmarks of the sm_100a tensor path that DESIGN.md section 7.1 argues from (csrc/microbench.cu, debug library
only): the latency of a short dependent chain of tcgen05.mma and the tcgen05.ld throughput beside running MMAs.  The
asserts are loose sanity bounds; the printed table (`-s`) is what profiles/r2_microbench.txt keeps."""
import ctypes as C

import pytest

import paper_2606_27216_b200 as hm
from paper_2606_27216_b200 import build as B

pytestmark = pytest.mark.gpu


def _lib():
    lib = C.CDLL(B.build_debug())
    lib.himuon_debug_microbench.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_longlong)]
    lib.himuon_debug_microbench.restype = C.c_int
    return lib


def _run(lib, which, param):
    out = (C.c_longlong * 2)()
    assert lib.himuon_debug_microbench(which, param, out) == 0
    return out[0], out[1]


def test_mma_chain_latency_is_a_fixed_cost_plus_throughput():
    lib = _lib()
    print()
    for which, N in ((0, 128), (1, 64)):
        cyc = {n: _run(lib, which, n)[0] for n in (1, 2, 4, 8, 16, 32, 64)}
        slope = (cyc[64] - cyc[32]) / 32.0
        fixed = cyc[8] - 8 * slope
        for n, c in cyc.items():
            print(f"tcgen05.mma 128x{N}x16 (A in TMEM), {n:2d} per commit: {c:5d} cycles from issue to commit seen")
        print(f"  -> {slope:.1f} cycles per MMA + {fixed:.0f} fixed")
        assert abs(slope - N / 2) < 0.15 * N / 2        # N / 2 cycles per K = 16 step: the full tensor rate
        assert 250 < fixed < 900                        # ... and several hundred cycles before the first result is visible


def test_tmem_read_throughput_beside_running_mmas():
    lib = _lib()
    passes = 2000
    print()
    for which, label in ((2, "alone"), (3, "with MMAs running")):
        cyc, prods = _run(lib, which, passes)
        bpc = passes * 65536 / cyc
        print(f"8 warps reading a 64 KB accumulator (tcgen05.ld.x16) {label}: {cyc / passes:.0f} cycles per pass, "
              f"{bpc:.0f} B per cycle and SM" + (f"; {prods} products of 8 MMAs completed meanwhile ({cyc / max(prods, 1):.0f} cycles each)" if which == 3 else ""))
        assert bpc > 300                                # nowhere near a bound on the epilogues (64 KB per phase)
