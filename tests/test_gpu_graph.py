"""himuon_step under CUDA stream capture: a bound plan whose work list is resident in its workspace issues nothing but
kernel launches (the large-tile path passes its tensor maps by value), so a whole optimizer step - one launch at
T <= 256, seventeen per sub-batch at T = 512 - can be captured once and replayed.  Replays must reproduce the eager
steps bit for bit (same kernels, same launch order, fixed summation orders)."""
import pytest
import torch

import himuon_inputs as I
import paper_2606_27216_b200 as hm

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _state(spec):
    Ws, Gs, Ms = [], [], []
    for i in range(len(spec.layers)):
        W, G, M = I.make_layer_tensors(spec, i, dtype=torch.bfloat16, device=DEV)
        Ws.append(W); Gs.append(G); Ms.append(M)
    return Ws, Gs, Ms


@pytest.mark.parametrize("T", [32, 128, 256, 512])
def test_step_replayed_from_a_cuda_graph_equals_eager(T):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    spec = I.gpt2_xl_spec(n_blocks=1)                    # 1600-wide layers: ragged at every T >= 128
    hp = hm.HParams(K=5, eps=1e-7, beta=0.95, nesterov=True, lr=0.02, wd=0.01, scale_c=0.2)
    # eager: three steps
    We, Ge, Me = _state(spec)
    plan_e = hm.Plan.from_tensors(We, Ge, Me, T).bind()
    for _ in range(3):
        plan_e.step(hp)
    torch.cuda.synchronize()
    plan_e.destroy()
    # captured: one eager step (loads the kernels, configures shared memory), then the step captured and replayed twice
    Wg, Gg, Mg = _state(spec)
    plan_g = hm.Plan.from_tensors(Wg, Gg, Mg, T).bind()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        plan_g.step(hp, stream=s)
        s.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            plan_g.step(hp, stream=s)
    torch.cuda.synchronize()
    # capturing does not execute: so far ONE step has run on the captured state
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    plan_g.destroy()
    for a, b in zip(We + Me, Wg + Mg):
        assert torch.equal(a, b)
        assert bool(torch.isfinite(a.float()).all())
