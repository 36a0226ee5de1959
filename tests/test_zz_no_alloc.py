"""mesh_attn_forward_static (include/mesh_attn.h; csrc/no_alloc.cu): the forward for callers that cannot allocate device
memory -- its partial (O, lse) scratch is a 32 MiB device array built into the library -- against the existing path
(mesh_attn_forward with caller-owned partials; Alg.2 l.3-6), on calls in a row that SHARE the array:

  call 1: a causal, striped, GQA plan (a = b = 2) after the array was filled with NaNs;
  call 2: a plan of another geometry (head_dim 64, a = 2, b = 1) straight after it: the array holds call 1's partials;
  call 3: the first plan again on other inputs: the array holds call 2's.

Each result is compared with the existing path's on the same inputs, within BASELINE.json's forward tolerances (the two run the
same kernels, so the difference printed is 0), and call 1 with the fp64 oracle on sampled rows.  Also: a plan beyond the limit is
refused with both byte counts in the error and launches nothing; the calls leave the device's free memory unchanged; the call
is captured into a CUDA graph and replayed (the use it exists for).

The file sorts last on purpose (pytest -x at the round's end: a failure here hides no other test); it passes alone in a fresh
process and after the other tests (the array is shared with nothing else)."""
import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.test_gpu_forward import check_against_oracle, sample_rows

pytestmark = pytest.mark.gpu

TOL_O_MAX, TOL_O_MEAN, TOL_LSE = 1e-2, 1e-3, 1e-3   # tests/test_gpu_forward.py


def _existing_path(plan, w, inp):
    from paper_2512_20968_b200 import Buffers

    buf = Buffers(plan, w, backward=False)
    plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
    torch.cuda.synchronize()
    return buf.O, buf.lse


def _compare(tag, O, lse, O_ref, lse_ref):
    assert torch.isfinite(O).all(), f"{tag}: non-finite output (a partial the call did not write itself?)"
    assert torch.equal(torch.isfinite(lse), torch.isfinite(lse_ref))
    fin = torch.isfinite(lse_ref)
    dO = (O - O_ref).abs()
    dl = (lse[fin] - lse_ref[fin]).abs().max().item() if fin.any() else 0.0
    print(f"{tag}: max|dO| {dO.max().item():.3e} mean|dO| {dO.mean().item():.3e} max|dLSE| {dl:.3e} "
          f"bit-identical {torch.equal(O, O_ref) and torch.equal(lse, lse_ref)}")
    assert dO.max().item() <= TOL_O_MAX and dO.mean().item() <= TOL_O_MEAN and dl <= TOL_LSE, tag


def test_forward_static_matches_forward_on_calls_in_a_row(oracle):
    from paper_2512_20968_b200 import plan_for

    wa = W.Workload("static_a", 21, True, 2, 2, 1, 4096, 8, 4, 128, seq_layout="striped")
    wb = W.Workload("static_b", 22, False, 2, 1, 1, 2048, 4, 4, 64, backward=False)
    wc = W.Workload("static_c", 23, True, 2, 2, 1, 4096, 8, 4, 128, seq_layout="striped")    # wa's geometry, other inputs
    pa, pb = plan_for(wa), plan_for(wb)
    ia, ib, ic = (W.make_inputs(w, "cuda", which=("q", "k", "v")) for w in (wa, wb, wc))
    refs = [_existing_path(pa, wa, ia), _existing_path(pb, wb, ib), _existing_path(pa, wc, ic)]

    need_a, cap = pa.forward_static_limits()
    need_b, _ = pb.forward_static_limits()
    assert cap == 32 << 20 and 0 < need_b < need_a <= cap, (need_a, need_b, cap)

    out = [(torch.full_like(O, float("nan")), torch.full_like(lse, float("nan"))) for O, lse in refs]
    pa.forward_static_poison()                              # every partial the first call reads must be its own
    pa.forward_static(ia["q"], ia["k"], ia["v"], *out[0])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]                    # the library's module (and its array) is loaded by now
    pb.forward_static(ib["q"], ib["k"], ib["v"], *out[1])   # same stream, straight after: finds call 1's partials
    pa.forward_static(ic["q"], ic["k"], ic["v"], *out[2])   # finds call 2's
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "a forward_static call changed the device's free memory"
    pa.health()
    pb.health()
    for tag, (O, lse), (O_ref, lse_ref) in zip(("call 1 (poisoned array)", "call 2 (other geometry)", "call 3 (other inputs)"), out, refs):
        _compare("forward_static " + tag, O, lse, O_ref, lse_ref)

    # call 1 against the fp64 oracle on sampled rows of every partition (the existing path's own bar)
    rows = sample_rows(wa, 4, np.random.default_rng(2100))
    check_against_oracle(oracle, wa, ia, out[0][0][0].cpu().numpy(), out[0][1][0].cpu().numpy(), rows=rows)


def test_forward_static_refuses_plans_beyond_the_array():
    from paper_2512_20968_b200 import launch_count, plan_for
    from paper_2512_20968_b200.binding import MeshAttnError

    w = W.Workload("static_big", 24, False, 2, 2, 1, 16384, 8, 8, 128)      # a * a * L * Hq * D * 4 = 64 MiB of partial_O
    plan = plan_for(w)
    need, cap = plan.forward_static_limits()
    assert need > cap
    inp = W.make_inputs(w, "cuda", which=("q", "k", "v"))
    O = torch.zeros((w.batch, w.seq_total, w.heads_q, w.head_dim), dtype=torch.float32, device="cuda")
    lse = torch.zeros((w.batch, w.heads_q, w.seq_total), dtype=torch.float32, device="cuda")
    n0 = launch_count()
    with pytest.raises(MeshAttnError) as e:
        plan.forward_static(inp["q"], inp["k"], inp["v"], O, lse)
    assert str(need) in str(e.value) and str(cap) in str(e.value), str(e.value)
    torch.cuda.synchronize()
    assert launch_count() == n0 and not O.any() and not lse.any()          # nothing was launched, nothing written


def test_forward_static_under_cuda_graph_capture():
    """The use the entry point is for: it is captured into a CUDA graph (no allocation, no host synchronisation, nothing on the
    default stream; the per-launch 4-byte memset of the work-item counter and the cluster launches are capturable) and the
    replays give the eager result bit for bit, also after the inputs were changed in place."""
    from paper_2512_20968_b200 import plan_for

    w = W.Workload("static_graph", 25, True, 2, 2, 1, 2048, 4, 4, 128, seq_layout="striped")
    plan = plan_for(w)
    inp = W.make_inputs(w, "cuda", which=("q", "k", "v"))
    O_ref, lse_ref = _existing_path(plan, w, inp)
    O, lse = torch.full_like(O_ref, float("nan")), torch.full_like(lse_ref, float("nan"))
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        plan.forward_static(inp["q"], inp["k"], inp["v"], O, lse, stream=side)      # warm-up: attributes, occupancy query, scratch address
    side.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        plan.forward_static(inp["q"], inp["k"], inp["v"], O, lse, stream=torch.cuda.current_stream())
    for rep in range(2):
        O.fill_(float("nan"))
        lse.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(O, O_ref) and torch.equal(lse, lse_ref), rep
    other = W.make_inputs(W.Workload("static_graph2", 26, True, 2, 2, 1, 2048, 4, 4, 128, seq_layout="striped"), "cuda", which=("q", "k", "v"))
    O2_ref, lse2_ref = _existing_path(plan, w, other)
    for name in ("q", "k", "v"):
        inp[name].copy_(other[name])                       # same buffers, new contents
    graph.replay()
    torch.cuda.synchronize()
    plan.health()
    assert torch.equal(O, O2_ref) and torch.equal(lse, lse2_ref)
