"""GPU parity of the Mesh-USP lanes: with usp_lanes = U every lane runs
Mesh-Attention on 1/U of the heads, so the result must be the same attention -- checked against the fp64 oracle
(BASELINE.json tolerances) and, for the forward, bit for bit against the one-lane plan (the per-(row, head)
arithmetic does not depend on which lane runs it).  Also: the per-kernel calls address simulated GPU g of n*U and
Q group q of b*U, and refuse ranges that cross a lane."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.test_gpu_backward import all_pairs, check_grads, check_invariants
from tests.test_gpu_forward import check_against_oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("U,batch,layout", [(2, 1, 0), (4, 2, 0), (2, 2, 1)])
def test_lanes_match_oracle_and_single_lane(oracle, U, batch, layout):
    from paper_2512_20968_b200 import Buffers, plan_for
    from paper_2512_20968_b200.binding import Q_PARTIAL_O_BYTES

    # causal GQA (16 query heads over 4 KV heads), 2 x 2 mesh, striped
    w = replace(W.scaled_down(W.C4, 256, heads_q=16), batch=batch, a=2, b=2, seq_total=4 * 256)
    inp = W.make_inputs(w, "cuda")
    if layout == 1:
        run_inp = {k: v.permute(0, 2, 1, 3).contiguous() for k, v in inp.items()}
    else:
        run_inp = inp

    def run(lanes):
        plan = plan_for(w, usp_lanes=lanes, tensor_layout=layout)
        buf = Buffers(plan, w, backward=True)
        if layout == 1:
            for name in ("O", "dQ", "dK", "dV"):
                t = getattr(buf, name)
                setattr(buf, name, torch.empty_like(t.permute(0, 2, 1, 3).contiguous()))
        for t in (buf.O, buf.lse, buf.dQ, buf.dK, buf.dV):
            t.fill_(float("nan"))
        plan.forward(run_inp["q"], run_inp["k"], run_inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
        plan.backward(run_inp["q"], run_inp["k"], run_inp["v"], buf.O, run_inp["do"], buf.lse, buf.bwd_ws, buf.dQ, buf.dK, buf.dV)
        torch.cuda.synchronize()
        if layout == 1:
            for name in ("O", "dQ", "dK", "dV"):
                setattr(buf, name, getattr(buf, name).permute(0, 2, 1, 3).contiguous())
        return plan, buf

    p1, b1 = run(1)
    pU, bU = run(U)
    assert pU.query(Q_PARTIAL_O_BYTES) * U == p1.query(Q_PARTIAL_O_BYTES)
    assert torch.equal(bU.O, b1.O) and torch.equal(bU.lse, b1.lse)
    assert torch.equal(bU.bwd_ws, b1.bwd_ws)
    for x, y in ((bU.dQ, b1.dQ), (bU.dK, b1.dK), (bU.dV, b1.dV)):
        assert (x - y).abs().max().item() <= 1e-3            # atomics: the summation order is run-dependent
    rows = np.arange(0, w.seq_total, 5)
    for bi in range(batch):
        check_against_oracle(oracle, w, inp, bU.O[bi].cpu().numpy(), bU.lse[bi].cpu().numpy(), rows=rows, batch_index=bi)
        qrows, qheads = all_pairs(rows, range(w.heads_q))
        krows, kheads = all_pairs(rows, range(w.heads_kv))
        check_grads(oracle, w, inp, bU, qrows, qheads, krows, kheads, bi=bi)
        check_invariants(w, inp, bU, bi=bi)


def test_per_kernel_calls_address_lanes(oracle):
    from paper_2512_20968_b200 import Buffers, plan_for
    from paper_2512_20968_b200.binding import EINVAL, MeshAttnError

    U = 2
    w = replace(W.scaled_down(W.C2, 128, heads_q=4), a=2, b=2, seq_total=4 * 128)
    inp = W.make_inputs(w, "cuda")
    plan = plan_for(w, usp_lanes=U)
    buf = Buffers(plan, w, backward=False)
    buf.O.fill_(float("nan"))
    # waves in reverse order, one (lane, Q group) at a time
    for wave in reversed(range(w.b * U)):
        lane, r = divmod(wave, w.b)
        plan.tile_fwd(lane * w.n + r * w.a, w.a, inp["q"], inp["k"], inp["v"], buf.partial_O, buf.partial_lse)
        plan.merge(wave, buf.partial_O, buf.partial_lse, buf.O, buf.lse)
    torch.cuda.synchronize()
    check_against_oracle(oracle, w, inp, buf.O[0].cpu().numpy(), buf.lse[0].cpu().numpy())
    for bad in ((w.n - 1, 2), (w.n * U - 1, 2), (w.n * U, 1)):           # crossing a lane / past the last lane
        with pytest.raises(MeshAttnError) as e:
            plan.tile_fwd(bad[0], bad[1], inp["q"], inp["k"], inp["v"], buf.partial_O, buf.partial_lse)
        assert e.value.status == EINVAL
    with pytest.raises(MeshAttnError):
        plan.merge(w.b * U, buf.partial_O, buf.partial_lse, buf.O, buf.lse)
