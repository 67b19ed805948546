"""`python bench.py --suite`: the per-config / per-T table behind BASELINE.json's metric
("HiMuon step ms & tiled-NS TFLOP/s (% of roofline) per model shape, per T"), one JSON line per row.

Rows: full steps on the GPT-2-small / GPT-2-XL / Llama-3-8B-shaped parameter sets (configs 2, 4, 5), the
tile-size sweep of Phi_{K,T} on the two config-3 matrices, and - as context, not as targets - a full-matrix
Phi_K through cuBLAS (torch.matmul, bf16 operands, fp32 accumulate) on the same config-3 matrices.
Every row: median of `--steps` launches timed with CUDA events after >= 3 warm-up launches; inputs of the
small configs are rotated over enough independent copies to exceed L2 (126 MB), and the row says so.
"""
from __future__ import annotations

import json
import statistics

import torch

import himuon_inputs as I

L2_BYTES = 126 << 20


def _time(fn, steps, warmup=3):
    for _ in range(max(3, warmup)):
        fn(0)
    torch.cuda.synchronize()
    ts = []
    for i in range(steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn(i)
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return statistics.median(ts), min(ts)


def _roof(flops, nbytes, pk):
    t_tensor = flops / (pk["bf16_sustained"] * 1e12)
    t_hbm = nbytes / (pk["hbm_gbs"] * 1e9)
    return ("tensor" if t_tensor >= t_hbm else "hbm"), max(t_tensor, t_hbm) * 1e3


def _emit(row):
    print(json.dumps(row), flush=True)


def _step_rows(args, hm, pk, dev):
    from bench import spec_of, algorithmic_flops, make_inputs
    hp = hm.HParams(K=args.K, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    AUTO, FP8 = hm.HIMUON_PATH_AUTO, hm.HIMUON_PATH_FP8
    for name, T, cap, path in (("gpt2-small", 128, 2048, AUTO), ("gpt2-xl", 128, 256, AUTO), ("llama3-8b", 128, 2048, AUTO),
                               ("llama3-8b", 16, 2048, AUTO), ("llama3-8b", 32, 2048, AUTO),
                               ("llama3-8b", 64, 2048, AUTO), ("llama3-8b", 256, 2048, AUTO), ("llama3-8b-sched", 128, 2048, AUTO),
                               ("llama3-8b", 512, 2048, AUTO), ("llama3-8b", 1 << 20, 2048, AUTO),
                               ("llama3-8b", (128, 256), 2048, AUTO), ("llama3-8b", (256, 64), 2048, AUTO),   # rectangular (T_h, T_w)
                               ("llama3-8b", 128, 2048, FP8), ("llama3-8b", 256, 2048, FP8)):   # opt-in e4m3 operands
        spec = spec_of(name)
        Tw = None
        if isinstance(T, tuple):                                            # tile-shape study
            T, Tw = T
        row = {"row": "step", "workload": name, "T": T, "cap_mb": cap}
        if Tw:
            row["T_w"] = Tw
        if path == FP8:
            row["path"] = "fp8 (e4m3 operands; reduced precision; peak = bf16 peak x 2)"
        try:
            n_sets = max(1, -(-2 * L2_BYTES // (10 * spec.n_elements)))     # rotate copies until > 2 x L2
            sets = [make_inputs(spec, dev) for _ in range(n_sets)]
            Tl = [l.T for l in spec.layers]
            plans = [hm.Plan.from_tensors(W, G, M, T, T_per_layer=Tl if any(Tl) else None, path=path,
                                          Tw_per_layer=[Tw] * len(W) if Tw else None,
                                          workspace_cap_bytes=cap << 20).bind() for (W, G, M) in sets]
            if Tw:      # Gram matrix on the short side s of the tile: (4 s^2 l + 2 s^3) K flops per s x l tile
                sh, lg = min(T, Tw), max(T, Tw)
                flops = float(sum((4.0 * sh + 2.0 * sh * sh / lg) * args.K * l.H * l.W for l in spec.layers))
            else:
                flops = algorithmic_flops(spec, T, args.K) if T <= 512 else float(sum(
                    6.0 * args.K * min(l.H, l.W) * l.H * l.W for l in spec.layers))   # full matrix: Gram on the short side
            med, best = _time(lambda i: plans[i % n_sets].step(hp), args.steps if (T <= 256 and not Tw) else 2)
            bound, roof_ms = _roof(flops, 10.0 * spec.n_elements,
                                   dict(pk, bf16_sustained=2 * pk["bf16_sustained"]) if path == FP8 else pk)
            row.update({"ms": round(med, 4), "ms_min": round(best, 4), "tflops": round(flops / med / 1e9, 2),
                        "gbs": round(10.0 * spec.n_elements / med / 1e6, 1), "bound": bound,
                        "roofline_ms": round(roof_ms, 4), "frac": round(roof_ms / med, 4), "tiles": plans[0].n_tiles,
                        "chunks": plans[0].n_chunks, "workspace_bytes": plans[0].workspace_bytes,
                        "input_sets_rotated": n_sets})
            del plans, sets
        except Exception as e:                                             # e.g. a tile size with no kernel yet
            row["unavailable"] = f"{type(e).__name__}: {e}"
        torch.cuda.empty_cache()
        _emit(row)


def _cublas_full_phi(G, K, a, b, c):
    """Context line: full-matrix NS through cuBLAS (bf16 operands, fp32 accumulate)."""
    X = G.float()
    X = (X / (X.norm() + 1e-7)).to(torch.bfloat16)
    tr = X.shape[0] > X.shape[1]
    if tr:
        X = X.t().contiguous()
    for _ in range(K):
        A = X @ X.t()
        B = torch.addmm(A, A, A, beta=b, alpha=c)
        X = torch.addmm(X, B, X, beta=a, alpha=1.0)
    return X.t() if tr else X


def _sweep_rows(args, hm, pk, dev):
    hp = hm.HParams(K=args.K, eps=1e-7)
    for (H, W) in ((4096, 4096), (4096, 11008)):
        n_sets = max(1, -(-2 * L2_BYTES // (4 * H * W)))
        Gs = [I.row_scaled_gaussian(H, W, seed_cfg=2, layer_index=i, dtype=torch.bfloat16, device=dev) for i in range(n_sets)]
        Us = [torch.empty_like(g) for g in Gs]
        for T in (16, 32, 64, 128, 256, 512):
            row = {"row": "phi_sweep", "workload": f"{H}x{W} bf16 row-scaled gaussian (config 3)", "T": T}
            try:
                plans = [hm.Plan.from_tensors([u], [g], None, T).bind() for u, g in zip(Us, Gs)]
                flops = 6.0 * args.K * T * H * W
                med, best = _time(lambda i: plans[i % n_sets].phi(hp), args.steps)
                bound, roof_ms = _roof(flops, 4.0 * H * W, pk)
                row.update({"ms": round(med, 4), "ms_min": round(best, 4), "tflops": round(flops / med / 1e9, 2),
                            "gbs": round(4.0 * H * W / med / 1e6, 1), "bound": bound, "roofline_ms": round(roof_ms, 4),
                            "frac": round(roof_ms / med, 4), "input_sets_rotated": n_sets})
            except Exception as e:
                row["unavailable"] = f"{type(e).__name__}: {e}"
            _emit(row)
        a, b, c = hm.NS_COEFFS
        med, best = _time(lambda i: _cublas_full_phi(Gs[i % n_sets], args.K, a, b, c), args.steps)
        r = min(H, W)
        flops = args.K * (2.0 * r * r * max(H, W) * 2 + 2.0 * r * r * r)
        _emit({"row": "context_cublas_full_matrix_phi", "workload": f"{H}x{W}", "ms": round(med, 4), "ms_min": round(best, 4),
               "tflops_executed": round(flops / med / 1e9, 2), "note": "torch.matmul/addmm bf16 (cuBLAS), not the tiled method"})
        del Gs, Us
        torch.cuda.empty_cache()


def run_suite(args):
    import paper_2606_27216_b200 as hm
    from bench import peaks
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    pk = peaks()
    _emit({"row": "peaks", **pk})
    _sweep_rows(args, hm, pk, dev)
    _step_rows(args, hm, pk, dev)
    _emit({"row": "context_paper", "note": "paper timings are on other hardware (A40 / H100, PAPER.md section 6); see BASELINE.md"})
