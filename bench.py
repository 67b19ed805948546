#!/usr/bin/env python
"""Benchmark of the HiMuon hot path on B200 (contract: see the task statement / DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload llama3-8b|gpt2-xl|gpt2-small] [--T 128]
    python bench.py --impl reference ...        # the float64 oracle timed on the host cores
    python bench.py --suite                     # per-config / per-T table (JSON lines), context lines included

One "step" = one pass of the whole hot path (plan already built; momentum -> tile -> normalise ->
K Newton-Schulz steps -> untile -> scaled, weight-decayed write) over one parameter set of seeded
synthetic gradients.  Default workload: BASELINE.json configs[4], the Llama-3-8B-shaped parameter set
(the configuration the north-star target is quoted on), T = 128, K = 5, bf16 storage.
Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

import himuon_inputs as I

METRIC = "himuon_step_tiled_ns_tflops"
UNIT = "TFLOP/s"


def spec_of(name: str):
    if name == "llama3-8b":
        return I.llama3_8b_spec()
    if name == "llama3-8b-sched":
        return I.llama3_8b_spec(schedule=True)
    if name == "gpt2-xl":
        return I.gpt2_xl_spec()
    if name == "gpt2-small":
        return I.gpt2_small_spec()
    raise SystemExit(f"unknown workload {name}")


def algorithmic_flops(spec, T_default: int, K: int) -> float:
    """6*K*T*H*W per matrix (Eq. 4.5; BASELINE.json north_star; reading Q16)."""
    return float(sum(6.0 * K * (l.T or T_default) * l.H * l.W for l in spec.layers))


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "bf16_burst": d["bf16_tflops"], "bf16_sustained": d["bf16_tflops_sustained"],
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.proc = gpu_index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.gpu)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ----------------------------------------------------------------------------- oracle legs (CPU)

def oracle_sample_run(spec, T: int, hp, n_tiles: int, seed: int = 1234):
    """Time the float64 oracle (as it stands) on a bounded sample of the workload: `n_tiles` T x T
    tiles cut from freshly drawn layers of the parameter set, one full Algorithm-4.1 step each.
    Returns (seconds, flops, cores)."""
    from oracle import himuon_oracle as O
    ohp = O.HParams(lr=hp.lr, beta=hp.beta, nesterov=bool(hp.nesterov), wd=hp.wd, K=hp.K, a=hp.a, b=hp.b, c=hp.c,
                    eps=hp.eps, scale_c=hp.scale_c)
    # draw one T-row strip of a layer per sample group (same recipe as the GPU inputs)
    tiles, li = [], 0
    while len(tiles) < n_tiles:
        l = spec.layers[li % len(spec.layers)]
        Tl = l.T or T
        cols = min(l.W, 8 * Tl)
        G = I.lowrank_plus_noise(Tl, cols, spec.rank, seed_cfg=spec.seed_cfg, layer_index=li, tensor_id=I.TENSOR_G)
        M = I.lowrank_plus_noise(Tl, cols, spec.rank, seed_cfg=spec.seed_cfg, layer_index=li, tensor_id=I.TENSOR_M)
        W = I.gaussian(Tl, cols, seed_cfg=spec.seed_cfg, layer_index=li, tensor_id=I.TENSOR_W, dtype=torch.bfloat16, scale=0.02)
        for c in range(cols // Tl):
            sl = slice(c * Tl, (c + 1) * Tl)
            tiles.append((I.to_f64_numpy(W[:, sl]), I.to_f64_numpy(G[:, sl]), I.to_f64_numpy(M[:, sl]), Tl))
        li += 1
    tiles = tiles[:n_tiles]
    t0 = time.perf_counter()
    flops = 0.0
    for (W, G, M, Tl) in tiles:
        O.step(W, G, M, ohp, Tl)   # a T x T block at tile size T is exactly one tile (R = C = 1)
        flops += 6.0 * hp.K * Tl * Tl * Tl
    dt = time.perf_counter() - t0
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = 1
    return dt, flops, cores


# ----------------------------------------------------------------------------- GPU arm

def make_inputs(spec, device):
    Ws, Gs, Ms = [], [], []
    for i in range(len(spec.layers)):
        W, G, M = I.make_layer_tensors(spec, i, dtype=torch.bfloat16, device=device)
        Ws.append(W); Gs.append(G); Ms.append(M)
    return Ws, Gs, Ms


def run_gpu(args):
    import paper_2606_27216_b200 as hm
    rank, world, local = dist_env()
    if args.gpus != world:
        if world == 1 and args.gpus > 1:
            raise SystemExit("launch multi-GPU runs with torch.distributed.run (one rank per GPU)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    spec = spec_of(args.workload)
    if args.blocks:
        per_block = {"llama3-8b": 7, "llama3-8b-sched": 7, "gpt2-xl": 6, "gpt2-small": 6}[args.workload]
        spec.layers = spec.layers[: per_block * args.blocks]
        spec.name += f"[first {args.blocks} blocks]"
    hp = hm.HParams(K=args.K, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    flops_job = algorithmic_flops(spec, args.T, args.K) * (1 if args.shard else world)
    if args.shard and world > 1:                              # strong scaling: whole matrices per rank, no collective
        from paper_2606_27216_b200.shard import shard_layers
        mine = shard_layers([l.H * l.W for l in spec.layers], world)[rank]
        spec.layers = [spec.layers[i] for i in mine]
    Ws, Gs, Ms = make_inputs(spec, dev)                       # default (weak scaling): every rank owns a full parameter set
    Tl = [l.T for l in spec.layers]
    path = hm.HIMUON_PATH_FP8 if args.path == "fp8" else hm.HIMUON_PATH_AUTO
    plan = hm.Plan.from_tensors(Ws, Gs, Ms, args.T, T_per_layer=Tl if any(Tl) else None, path=path,
                                workspace_cap_bytes=args.cap_mb << 20).bind()
    flops = algorithmic_flops(spec, args.T, args.K)
    n_elem = spec.n_elements
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        plan.step(hp)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = hm.himuon_launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.profiler.start()       # no-op unless run under `ncu --profile-from-start off`
    t_begin.record(stream)
    for k in range(args.steps):
        evs[k][0].record(stream)
        plan.step(hp)
        evs[k][1].record(stream)
    t_end.record(stream)
    barrier()
    torch.cuda.profiler.stop()
    launches = hm.himuon_launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = t_begin.elapsed_time(t_end)
    per_step = [a.elapsed_time(b) for a, b in evs]
    if world > 1:
        import torch.distributed as dist
        t = torch.tensor([total_ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = flops_job / (ms_per_step * 1e-3) / 1e12

    # ---- e2e: same metric through the public API with HOST buffers (gradients in, weights out)
    e2e = run_e2e(args, hm, spec, plan, hp, Ws, Gs, flops, world, dev, barrier)

    if rank != 0:
        return
    pk = peaks()
    # dominant kernel = the fused step kernel of the plan-wide tile size (one launch per chunk)
    kname = {16: "himuon_warp_kernel", 32: "himuon_warp_kernel", 64: "himuon_tc64_kernel", 128: "himuon_tc128_kernel",
             256: "himuon_tc256_kernel"}.get(args.T, "himuon_simt_kernel")
    if args.path == "fp8":                                    # e4m3 peak = measured bf16 peak x the nominal 2:1 ratio
        kname = "himuon_tc256_kernel<F8>" if args.T == 256 else "himuon_tc128_kernel<F8>"
        pk = dict(pk, bf16_sustained=2 * pk["bf16_sustained"], bf16_burst=2 * pk["bf16_burst"],
                  source=pk["source"] + " x2 (nominal fp8:bf16 ratio)")
    kern_ms = statistics.mean(per_step) / max(1, plan.n_chunks)
    bytes_step = 10.0 * n_elem
    t_tensor = flops / (pk["bf16_sustained"] * 1e12)
    t_hbm = bytes_step / (pk["hbm_gbs"] * 1e9)
    traffic, traffic_src = None, None
    for tp in ("r2_traffic.csv", "r1_traffic.csv"):           # newest ncu capture: DRAM bytes per element x elements per launch
        tpath = os.path.join(ROOT, "profiles", tp)
        if traffic is None and os.path.exists(tpath):
            for ln in open(tpath).read().splitlines()[1:]:
                f = ln.split(",")
                if f[0] == kname and int(f[1]) == args.T and not any(l.T for l in spec.layers):
                    traffic = float(f[5]) * n_elem / plan.n_chunks
                    traffic_src = f"ncu capture profiles/{tp} (dram bytes per element of a {f[2]}-element launch) x elements of this launch; not measured in this run"
    if t_tensor >= t_hbm:
        ach = flops / plan.n_chunks / (kern_ms * 1e-3) / 1e12
        roof = {"bound": "tensor", "achieved": round(ach, 2), "peak": pk["bf16_sustained"], "unit": "TFLOP/s",
                "frac": round(ach / pk["bf16_sustained"], 4), "traffic": traffic,
                "peak_kind": "sustained bf16, " + pk["source"], "frac_of_burst": round(ach / pk["bf16_burst"], 4)}
    else:
        ach = bytes_step / plan.n_chunks / (kern_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": round(ach, 1), "peak": pk["hbm_gbs"], "unit": "GB/s",
                "frac": round(ach / pk["hbm_gbs"], 4), "traffic": traffic, "peak_kind": "copy bandwidth, " + pk["source"]}
    roof.update({"traffic_source": traffic_src, "kernel": kname, "launch_ms": round(kern_ms, 4),
                 "tflops_achieved": round(flops / (ms_per_step * 1e-3) / 1e12, 2),
                 "hbm_gbs_achieved": round(bytes_step / (ms_per_step * 1e-3) / 1e9, 1),
                 "roofline_ms": round(max(t_tensor, t_hbm) * 1e3, 3)})
    cpu = run_cpu_baseline(args, spec, hp)
    context = {"cublas_full_matrix_phi": cublas_full_matrix_context(spec, args.K, dev), "paper": PAPER_CONTEXT,
               "cpu_oracle": "see cpu_baseline (float64 oracle on this box's host cores, same run)"}
    line = {"metric": METRIC, "value": round(value, 2), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": round(ms_per_step, 4), "higher_is_better": True,
            "scaling": "strong" if args.shard else "weak", "vs_baseline": None, "dtype": "fp8-e4m3 operands, fp32 state" if args.path == "fp8" else "bf16", "data": "synthetic",
            "config": {"workload": f"{spec.name}-shaped HiMuon step (BASELINE configs[4])" if spec.name.startswith("llama3-8b") else f"{spec.name}-shaped HiMuon step",
                       "layers": len(spec.layers), "elements": n_elem, "tiles": plan.n_tiles, "T": args.T, "K": args.K,
                       "chunks": plan.n_chunks, "workspace_bytes": plan.workspace_bytes, "cap_mb": args.cap_mb,
                       "l2": "inputs (%.1f GB) larger than L2" % (bytes_step / 1e9),
                       "state": "timed steps run back-to-back on the W and M the previous step wrote (no restore between steps)", "parallelism": (f"whole matrices sharded over {world} ranks" if args.shard else f"replicas x{world}") + ", no collective",
                       "gflop_per_step": round(flops / 1e9, 1)},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
            "context": context,
            "step_ms_median": round(statistics.median(per_step), 4), "step_ms_min": round(min(per_step), 4)}
    print(json.dumps(line))


def run_e2e(args, hm, spec, plan, hp, Ws, Gs, flops, world, dev, barrier):
    """Per step, over the WHOLE parameter set: H2D copy of every layer's gradient from pinned host memory,
    himuon_step, D2H read of every updated weight into pinned host memory - through the public API (one bound plan
    per group of layers), pipelined over three streams so that the copies of one group overlap the step of another
    (PCIe is full duplex).  Pinned host memory is a ring of group-sized slots bounded by --e2e-host-gb: with enough
    budget every group has its own slot; otherwise slots are reused round-robin within a step (groups sharing a slot
    receive the same gradient bits and overwrite each other's read-back - same bytes over the link, same kernels).
    Momentum buffers of this leg are separate zero-initialised tensors (the timed loop above keeps its own)."""
    per_group = max(1, {"gpt2": 6}.get(spec.name[:4], 7))          # one transformer block
    n_layers = len(Gs)
    groups = [list(range(a, min(a + per_group, n_layers))) for a in range(0, n_layers, per_group)]
    slot_bytes = max(sum(Gs[i].numel() * 2 for i in gr) for gr in groups)          # one G-in or W-out slot
    budget = int(args.e2e_host_gb * (1 << 30) / max(1, world))   # pinned host memory is shared by the ranks of a node
    n_slots = max(1, min(len(groups), budget // (2 * slot_bytes)))
    Tl = [l.T for l in spec.layers]
    plans = []
    for gr in groups:
        Ms_g = [torch.zeros_like(Gs[i]) for i in gr]
        plans.append(hm.Plan.from_tensors([Ws[i] for i in gr], [Gs[i] for i in gr], Ms_g, args.T,
                                          T_per_layer=[Tl[i] for i in gr] if any(Tl) else None,
                                          path=hm.HIMUON_PATH_FP8 if args.path == "fp8" else hm.HIMUON_PATH_AUTO).bind())
    hG = [torch.empty(slot_bytes // 2, dtype=torch.bfloat16, pin_memory=True) for _ in range(n_slots)]
    hW = [torch.empty(slot_bytes // 2, dtype=torch.bfloat16, pin_memory=True) for _ in range(n_slots)]

    def views(buf, gr):            # per-layer views of a slot
        out, off = [], 0
        for i in gr:
            n = Gs[i].numel()
            out.append(buf[off:off + n].view(Gs[i].shape))
            off += n
        return out

    for k, gr in enumerate(groups[:n_slots]):                     # seed the ring with this rank's gradients
        for v, i in zip(views(hG[k], gr), gr):
            v.copy_(Gs[i])
    steps = max(2, min(args.steps, 5))
    s_in, s_cmp, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
    ev_cmp_prev = [None] * len(groups)       # G of a group may be overwritten once the previous step of it is done
    ev_out_prev = [None] * len(groups)       # W of a group may be overwritten once its previous read-back is done

    def one():
        for k, gr in enumerate(groups):
            slot = k % n_slots
            with torch.cuda.stream(s_in):
                if ev_cmp_prev[k] is not None:
                    s_in.wait_event(ev_cmp_prev[k])
                for v, i in zip(views(hG[slot], gr), gr):
                    Gs[i].copy_(v, non_blocking=True)
                e_in = torch.cuda.Event(); e_in.record(s_in)
            with torch.cuda.stream(s_cmp):
                s_cmp.wait_event(e_in)
                if ev_out_prev[k] is not None:
                    s_cmp.wait_event(ev_out_prev[k])
                plans[k].step(hp, stream=s_cmp)
                e_c = torch.cuda.Event(); e_c.record(s_cmp)
            with torch.cuda.stream(s_out):
                s_out.wait_event(e_c)
                for v, i in zip(views(hW[slot], gr), gr):
                    v.copy_(Ws[i], non_blocking=True)
                e_o = torch.cuda.Event(); e_o.record(s_out)
            ev_cmp_prev[k], ev_out_prev[k] = e_c, e_o

    def join(stream):
        for s_ in (s_in, s_cmp, s_out):
            e = torch.cuda.Event(); e.record(s_); stream.wait_event(e)

    cur = torch.cuda.current_stream()
    one(); join(cur)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cur)
    for s_ in (s_in, s_cmp, s_out):
        s_.wait_event(e0)
    for _ in range(steps):
        one()
    join(cur)
    e1.record(cur)
    barrier()
    ms = e0.elapsed_time(e1) / steps
    if world > 1:
        import torch.distributed as dist
        t = torch.tensor([ms], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    nbytes = sum(g.numel() * 2 for g in Gs)
    ring = (f"every group has its own pinned slot ({n_slots} x 2 x {slot_bytes / 2**20:.0f} MiB)" if n_slots == len(groups) else
            f"ring of {n_slots} pinned slots of 2 x {slot_bytes / 2**20:.0f} MiB reused round-robin over {len(groups)} groups "
            f"(--e2e-host-gb {args.e2e_host_gb})")
    return {"value": round(world * flops / (ms * 1e-3) / 1e12, 3), "unit": UNIT, "ms_per_step": round(ms, 3),
            "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "steps": steps,
            "pipeline": f"{len(groups)} groups of layers (one plan each) over 3 streams: H2D | himuon_step | D2H",
            "workload": "full parameter set", "host_buffers": ring,
            "momentum": "separate zero-initialised M buffers for this leg; steps back-to-back on the mutated W, M",
            "link_gbs_each_way": round(nbytes / (ms * 1e-3) / 1e9, 1)}


def cublas_full_matrix_context(spec, K, dev):
    """Context line (north_star): full-matrix Phi_K (Muon's T = infinity) through cuBLAS
    (torch.matmul / addmm, bf16 operands, fp32 accumulation) on the SAME matrices' shapes: one matrix of each distinct
    shape is timed (median of 3 after 2 warm-ups, CUDA events) and multiplied by how often the shape occurs."""
    import paper_2606_27216_b200 as hm
    a, b, c = hm.NS_COEFFS
    shapes = {}
    for i, l in enumerate(spec.layers):
        shapes.setdefault((l.H, l.W), []).append(i)
    total_ms, flops, per_shape = 0.0, 0.0, []
    for (H, W), idx in shapes.items():
        G = I.lowrank_plus_noise(H, W, spec.rank, seed_cfg=spec.seed_cfg, layer_index=idx[0], tensor_id=I.TENSOR_G,
                                 dtype=torch.bfloat16, device=dev)

        def run():
            X = G.float()
            X = (X / (X.norm() + 1e-7)).to(torch.bfloat16)
            if H > W:
                X = X.t().contiguous()                    # work on the short side
            for _ in range(K):
                A = X @ X.t()
                B = torch.addmm(A, A, A, beta=b, alpha=c)
                X = torch.addmm(X, B, X, beta=a, alpha=1.0)
            return X

        ts = []
        for rep_ in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); run(); e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        ms = statistics.median(ts[2:])
        r, n = min(H, W), max(H, W)
        fl = K * (4.0 * r * r * n + 2.0 * r * r * r)
        per_shape.append({"shape": [H, W], "count": len(idx), "ms_each": round(ms, 3)})
        total_ms += ms * len(idx)
        flops += fl * len(idx)
        del G
    torch.cuda.empty_cache()
    return {"what": "cuBLAS full-matrix Phi_K (Muon, T = infinity) on the same matrix shapes: Phi only, no momentum / "
                    "update passes; one matrix per distinct shape timed, x count",
            "ms_per_parameter_set": round(total_ms, 2), "tflops_executed": round(flops / total_ms / 1e9, 1),
            "gflop_executed": round(flops / 1e9, 1), "per_shape": per_shape,
            "note": "context, not the target: a different (more expensive) map than the tiled one"}


PAPER_CONTEXT = [
    # the paper prints ratios, not absolute kernel times; quoted with their hardware, context only
    {"cite": "PAPER.md:374-380 (Fig. 7)", "hardware": "1x A40, bf16",
     "what": "SRAM-resident all-K-steps NS kernel vs PyTorch eager bmm loop, T=128, K=5, B_tile in {32,128,512,2048}",
     "value": "4-8x faster, largest at B_tile=2048"},
    {"cite": "PAPER.md:398-402 (Fig. 9a)", "hardware": "1x A40, bf16",
     "what": "optimizer step vs full-matrix Muon, 8 stacked Linear(H,H), T=512, K=5, H = 1024 / 2048 / 4096",
     "value": "tiled only 1.4x / 3.2x / 5.2x; with cross-layer batching 2.3x / 3.7x / 5.4x"},
    {"cite": "PAPER.md:355-370 (Fig. 6)", "hardware": "1x A40, bf16",
     "what": "per-layer tiled / full-matrix NS speedup at T=512, K=5, Qwen3 block-0 shapes",
     "value": "1.4-1.6x (0.6B), 1.4-2.9x (1.7B), 1.3-2.9x (4B)"},
    {"cite": "PAPER.md:341-349", "hardware": "4x A40 DDP / FSDP, bf16 mixed",
     "what": "end-to-end training step time, T = inf -> 512 -> 128 schedule",
     "value": "Qwen3-0.6B 3.80 -> 3.62 s; 1.7B 6.72 -> 6.16 s; 4B 17.55 -> 17.18 s"},
]


def run_cpu_baseline(args, spec, hp):
    n = args.cpu_tiles
    dt, fl, cores = oracle_sample_run(spec, args.T, hp, n)
    return {"value": round(fl / dt / 1e12, 6), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n} tiles of {args.T}x{args.T} (one Algorithm-4.1 step each) drawn with the {spec.name} recipe; "
                      f"{dt:.1f} s of float64 numpy", "seconds": round(dt, 2)}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step = a bounded sample."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import paper_2606_27216_b200 as hm   # HParams container only; no kernels are called on this arm
    spec = spec_of(args.workload)
    hp = hm.HParams(K=args.K, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    n = max(8, args.cpu_tiles // 8)
    for _ in range(args.warmup):
        oracle_sample_run(spec, args.T, hp, n)
    tot_t, tot_f, cores = 0.0, 0.0, 1
    for _ in range(args.steps):
        dt, fl, cores = oracle_sample_run(spec, args.T, hp, n)
        tot_t += dt; tot_f += fl
    v = tot_f / tot_t / 1e12
    line = {"impl": "reference", "metric": METRIC, "value": round(v, 6), "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(tot_t / args.steps * 1e3, 2),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{spec.name}-shaped HiMuon step, bounded sample of {n} tiles per step", "T": args.T, "K": args.K},
            "cpu_baseline": {"value": round(v, 6), "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{n} tiles of {args.T}x{args.T} per step, {args.steps} steps"},
            "e2e": {"value": round(v, 6), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="himuon", choices=["himuon", "reference"])
    ap.add_argument("--workload", default="llama3-8b")
    ap.add_argument("--T", type=int, default=128)
    ap.add_argument("--K", type=int, default=5)
    ap.add_argument("--path", default="auto", choices=["auto", "fp8"],
                    help="fp8: e4m3 operands in the Newton-Schulz products (T = 128 / 256 only; NOT the headline: reduced precision)")
    ap.add_argument("--cap-mb", type=int, default=2048)
    ap.add_argument("--cpu-tiles", type=int, default=16384)
    ap.add_argument("--e2e-host-gb", type=float, default=32.0, help="pinned host memory for the e2e leg (ring of group slots)")
    ap.add_argument("--blocks", type=int, default=0, help="truncate the parameter set to its first N transformer blocks (profiling only)")
    ap.add_argument("--shard", action="store_true", help="N > 1: split the parameter set over the ranks by whole matrices (strong scaling)")
    ap.add_argument("--suite", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.suite:
        from bench_suite import run_suite
        return run_suite(args)
    run_gpu(args)


if __name__ == "__main__":
    main()
