"""GPU parity of the GOO executor: the forward run task by task in the order of
the plan's step list -- chunk-granular tile launches C-i-j, device-to-device copies standing in for AG-KV / AG-Q / RS-Q
on a second stream, a barrier per step -- must give the attention of mesh_attn_forward (compared to tolerance: the
merge tree and the references of the bf16 roundings of P differ) and of the fp64 oracle, with and without the communication stand-ins."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.test_gpu_forward import check_against_oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("k_q,k_kv,order,causal", [(2, 2, "greedy", True), (3, 3, "greedy", False), (1, 1, "row_major", True),
                                                   (4, 2, "greedy", True)])
def test_executor_matches_forward_and_oracle(oracle, k_q, k_kv, order, causal):
    from paper_2512_20968_b200 import Buffers, plan_for
    from paper_2512_20968_b200 import binding as B

    L = 128 * k_q * k_kv
    base = W.C5 if causal else W.C2
    w = replace(W.scaled_down(base, L, heads_q=4), a=2, b=3, seq_total=6 * L, heads_kv=2, order=order, k_q=k_q, k_kv=k_kv)
    inp = W.make_inputs(w, "cuda")
    plan = plan_for(w)
    ref = Buffers(plan, w, backward=False)
    plan.forward(inp["q"], inp["k"], inp["v"], ref.O, ref.lse, ref.partial_O, ref.partial_lse)
    f32 = dict(dtype=torch.float32, device="cuda")
    part_O = torch.empty(plan.query(B.Q_GOO_PARTIAL_O_BYTES) * w.a // 4, **f32)
    part_lse = torch.empty(plan.query(B.Q_GOO_PARTIAL_LSE_BYTES) * w.a // 4, **f32)
    assert plan.query(B.Q_GOO_PARTIAL_O_BYTES) == k_kv * plan.query(B.Q_PARTIAL_O_BYTES)
    comm_ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    for comm_repeat, overlap in ((0, True), (2, True), (1, False)):
        O = torch.full_like(ref.O, float("nan"))
        lse = torch.full_like(ref.lse, float("nan"))
        part_O.fill_(float("nan"))
        part_lse.fill_(float("nan"))
        before = B.launch_count()
        for r in range(w.b):
            plan.forward_goo(r, inp["q"], inp["k"], inp["v"], O, lse, part_O, part_lse, comm_ws=comm_ws, comm_repeat=comm_repeat,
                             overlap=overlap)
        torch.cuda.synchronize()
        assert B.launch_count() - before == w.b * (k_q * k_kv + 1)            # one launch per compute task + the merge
        # P is rounded to bf16 relative to each task's own running max, so the two runs differ at bf16-operand level
        assert (O - ref.O).abs().max().item() <= 3e-3
        fin = torch.isfinite(ref.lse)
        assert torch.equal(torch.isfinite(lse), fin) and (lse[fin] - ref.lse[fin]).abs().max().item() <= 1e-4
        check_against_oracle(oracle, w, inp, O[0].cpu().numpy(), lse[0].cpu().numpy(), rows=np.arange(0, w.seq_total, 3))


def test_executor_argument_checks():
    from paper_2512_20968_b200 import Buffers, plan_for
    from paper_2512_20968_b200.binding import EINVAL, MeshAttnError

    w = replace(W.scaled_down(W.C2, 128, heads_q=2), a=2, b=2, seq_total=4 * 128)
    inp = W.make_inputs(w, "cuda")
    plan = plan_for(w)
    buf = Buffers(plan, w, backward=False)
    for kw in (dict(q_group=w.b), dict(q_group=0, comm_repeat=1)):             # past the last group; copies without a workspace
        with pytest.raises(MeshAttnError) as e:
            plan.forward_goo(kw.pop("q_group"), inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse, **kw)
        assert e.value.status == EINVAL


@pytest.mark.parametrize("k_q,k_kv,order,causal,hkv", [(2, 2, "greedy", True, 2), (3, 3, "greedy", False, 4), (1, 1, "row_major", True, 2),
                                                       (4, 2, "greedy", True, 1)])
def test_backward_executor_matches_backward(oracle, k_q, k_kv, order, causal, hkv):
    """mesh_attn_backward_goo: the backward step list run task by task (chunk-granular tile_bwd launches, copies standing in
    for AG-QOdO / AG-KV / RS-dQ / RS-dKV) accumulates the gradients of mesh_attn_backward: compared to the fused backward
    (only the order of the fp32 atomics differs) and, on sampled rows, to the fp64 oracle (2e-2 max abs)."""
    from paper_2512_20968_b200 import Buffers, plan_for
    from paper_2512_20968_b200 import binding as B
    from tests.util import torch_bits

    L = 128 * k_q * k_kv
    base = W.C5 if causal else W.C2
    w = replace(W.scaled_down(base, L, heads_q=4), a=2, b=3, seq_total=6 * L, heads_kv=hkv, order=order, k_q=k_q, k_kv=k_kv)
    inp = W.make_inputs(w, "cuda")
    plan = plan_for(w)
    ref = Buffers(plan, w, backward=True)
    plan.forward(inp["q"], inp["k"], inp["v"], ref.O, ref.lse, ref.partial_O, ref.partial_lse)
    plan.backward(inp["q"], inp["k"], inp["v"], ref.O, inp["do"], ref.lse, ref.bwd_ws, ref.dQ, ref.dK, ref.dV)
    comm_ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    steps = plan.steps(backward=True)
    n_compute = int((steps[:, 1] == B.TASK_C).sum())
    assert n_compute == k_q * k_kv
    for comm_repeat, overlap in ((0, True), (2, True), (1, False)):
        dQ, dK, dV = torch.zeros_like(ref.dQ), torch.zeros_like(ref.dK), torch.zeros_like(ref.dV)
        before = B.launch_count()
        for r in range(w.b):
            plan.backward_goo(r, inp["q"], inp["k"], inp["v"], inp["do"], ref.bwd_ws, dQ, dK, dV, comm_ws=comm_ws, comm_repeat=comm_repeat,
                              overlap=overlap)
        torch.cuda.synchronize()
        assert B.launch_count() - before == w.b * n_compute
        for name, got, want in (("dQ", dQ, ref.dQ), ("dK", dK, ref.dK), ("dV", dV, ref.dV)):
            assert torch.isfinite(got).all()
            err = (got - want).abs().max().item()
            assert err <= 1e-3 * max(1.0, want.abs().max().item()), f"{name}: {err:.3e} vs mesh_attn_backward"
    q, k, v, do = (torch_bits(inp[x][0]) for x in ("q", "k", "v", "do"))
    pos = oracle.positions(w.n, w.L, w.seq_layout)
    rng = np.random.default_rng(3)
    rows = rng.integers(0, w.seq_total, 64)
    heads = rng.integers(0, w.heads_q, 64).astype(np.int32)
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, rows, heads)
    assert np.abs(dQ[0].cpu().numpy()[rows, heads] - dq_ref).max() <= 2e-2
    krows = rng.integers(0, w.seq_total, 32)
    kheads = rng.integers(0, w.heads_kv, 32).astype(np.int32)
    dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, w.causal, pos, krows, kheads)
    assert np.abs(dK[0].cpu().numpy()[krows, kheads] - dk_ref).max() <= 2e-2
    assert np.abs(dV[0].cpu().numpy()[krows, kheads] - dv_ref).max() <= 2e-2
