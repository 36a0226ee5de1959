"""GPU parity of the per-rank calls (include/mesh_attn.h "per-rank calls"): the n ranks of a job are
played ONE AFTER THE OTHER on one B200 (no rank waits on another), each on tensors that hold only its gathered
partitions; the exchanges between them (AG-Q, AG-KV, RS-O, RS-dQ, RS-dKV) are index copies on the device.  The results
must equal the simulated-GPU path's (forward bit for bit: same kernels, same work lists, same merge order; backward up
to the order of the fp32 atomics) and the fp64 oracle's within BASELINE.json's tolerances."""
import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.test_gpu_forward import check_against_oracle, run_forward, sample_rows

pytestmark = pytest.mark.gpu


def play_ranks(plan, w, inp, backward=True):
    B, L, Hq, Hkv, D, a, b, n = w.batch, w.L, w.heads_q, w.heads_kv, w.head_dim, w.a, w.b, w.n
    f32 = dict(dtype=torch.float32, device="cuda")
    part = lambda t, p: t[:, p * L:(p + 1) * L]                                  # noqa: E731
    gather = lambda t, parts: torch.cat([part(t, int(p)) for p in parts], dim=1).contiguous()   # noqa: E731
    foot = [plan.footprint(g) for g in range(n)]
    # forward: AG-Q, AG-KV, rank_fwd
    loc, partials = [], []
    for g in range(n):
        iq, ikv = foot[g]
        Ql, Kl, Vl = gather(inp["q"], iq), gather(inp["k"], ikv), gather(inp["v"], ikv)
        pO = torch.full((a, B, L, Hq, D), float("nan"), **f32)
        pl = torch.full((a, B, Hq, L), float("nan"), **f32)
        plan.rank_fwd(g, Ql, Kl, Vl, pO, pl)
        loc.append((Ql, Kl, Vl))
        partials.append((pO, pl))
    # RS-O: rank u receives slot (index of u in the member's I^Q) from every member of its Q group, then merges
    O = torch.empty((B, n * L, Hq, D), **f32)
    lse = torch.empty((B, Hq, n * L), **f32)
    own = []
    for u in range(n):
        members = [int(x) for x in foot[u][0]]
        k_u = members.index(u)
        rO = torch.stack([partials[m][0][k_u] for m in members]).contiguous()
        rl = torch.stack([partials[m][1][k_u] for m in members]).contiguous()
        O_own = torch.full((B, L, Hq, D), float("nan"), **f32)
        lse_own = torch.full((B, Hq, L), float("nan"), **f32)
        plan.rank_merge(rO, rl, O_own, lse_own)
        # the same merge reading each partial where its producer wrote it (separate allocations stand in for peer memory)
        O_peer, lse_peer = torch.full_like(O_own, float("nan")), torch.full_like(lse_own, float("nan"))
        plan.rank_merge_peers([partials[m][0][k_u] for m in members], [partials[m][1][k_u] for m in members], O_peer, lse_peer)
        assert torch.equal(O_peer, O_own) and torch.equal(lse_peer, lse_own), "peer-memory merge differs from rank_merge"
        own.append((O_own, lse_own))
        part(O, u).copy_(O_own)
        lse[:, :, u * L:(u + 1) * L].copy_(lse_own)
    if not backward:
        return O, lse, None
    # backward: preprocess on the own rows; AG of dO and (delta, offset); rank_bwd; reduce-scatters as sums
    ws_own = []
    for u in range(n):
        ws = torch.empty((2, B, Hq, L), **f32)
        plan.rank_bwd_preprocess(own[u][0], part(inp["do"], u).contiguous(), own[u][1], ws)
        ws_own.append(ws)
    dQ = torch.zeros((B, n * L, Hq, D), **f32)
    dK = torch.zeros((B, n * L, Hkv, D), **f32)
    dV = torch.zeros((B, n * L, Hkv, D), **f32)
    grads_loc = []
    for g in range(n):
        iq, ikv = foot[g]
        Ql, Kl, Vl = loc[g]
        dOl = gather(inp["do"], iq)
        ws_loc = torch.cat([ws_own[int(u)] for u in iq], dim=3).contiguous()     # [2, B, Hq, a*L]
        dQl = torch.zeros((B, a * L, Hq, D), **f32)
        dKl = torch.zeros((B, b * L, Hkv, D), **f32)
        dVl = torch.zeros((B, b * L, Hkv, D), **f32)
        plan.rank_bwd(g, Ql, Kl, Vl, dOl, ws_loc, dQl, dKl, dVl)
        grads_loc.append((dQl, dKl, dVl))
    # RS-dQ / RS-dKV: rank u sums its slot of every member's local gradients, read where the members wrote them
    assert B == 1
    for u in range(n):
        q_members, kv_members = [int(x) for x in foot[u][0]], [int(x) for x in foot[u][1]]
        k_u, t_u = q_members.index(u), kv_members.index(u)
        for which, members, slot, dst in ((0, q_members, k_u, dQ), (1, kv_members, t_u, dK), (2, kv_members, t_u, dV)):
            own_sum = torch.empty_like(part(dst, u)[0])
            plan.rank_sum_peers([part(grads_loc[m][which], slot)[0] for m in members], own_sum)
            part(dst, u).copy_(own_sum)
    torch.cuda.synchronize()
    return O, lse, (dQ, dK, dV)


@pytest.mark.parametrize("base,L,hq,hkv", [(W.C2, 256, 2, 2), (W.C3, 512, 2, 2), (W.C4, 128, 8, 2)], ids=["C2s", "C3s", "C4s-gqa"])
def test_rank_calls_equal_simulated_gpus(oracle, base, L, hq, hkv):
    from paper_2512_20968_b200 import Buffers, plan_for

    w = W.scaled_down(base, L, heads_q=hq, heads_kv=hkv)
    inp = W.make_inputs(w, "cuda")
    prec = 1 if w.outlier else 0
    plan = plan_for(w, precision=prec)
    O, lse, grads = play_ranks(plan, w, inp)
    # the simulated-GPU path on the same plan
    buf = Buffers(plan, w, backward=True)
    plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
    plan.backward(inp["q"], inp["k"], inp["v"], buf.O, inp["do"], buf.lse, buf.bwd_ws, buf.dQ, buf.dK, buf.dV)
    torch.cuda.synchronize()
    assert torch.equal(O, buf.O), "forward O differs from the simulated-GPU path"
    assert torch.equal(lse, buf.lse), "forward lse differs from the simulated-GPU path"
    for name, got, ref in zip(("dQ", "dK", "dV"), grads, (buf.dQ, buf.dK, buf.dV)):
        assert torch.isfinite(got).all()
        err = (got - ref).abs().max().item()
        assert err <= 1e-3 * max(1.0, ref.abs().max().item()), f"{name}: {err:.3e} vs the simulated-GPU path"
    # and the oracle directly (forward rows of every partition)
    rows = sample_rows(w, 2, np.random.default_rng(5))
    check_against_oracle(oracle, w, inp, O[0].cpu().numpy(), lse[0].cpu().numpy(), rows=rows, heads=[0, hq - 1])


def test_rank_calls_gradients_against_oracle(oracle):
    """dQ rows and tail-key dK/dV of the played ranks against the fp64 oracle (gradient tolerance 2e-2 max abs)."""
    w = W.scaled_down(W.C4, 128, heads_q=4, heads_kv=2)
    inp = W.make_inputs(w, "cuda")
    from paper_2512_20968_b200 import plan_for
    from tests.util import torch_bits

    plan = plan_for(w)
    _, _, (dQ, dK, dV) = play_ranks(plan, w, inp)
    q, k, v, do = (torch_bits(inp[x][0]) for x in ("q", "k", "v", "do"))
    pos = oracle.positions(w.n, w.L, w.seq_layout)
    rng = np.random.default_rng(11)
    rows = rng.integers(0, w.seq_total, 96)
    heads = rng.integers(0, w.heads_q, 96).astype(np.int32)
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, rows, heads)
    assert np.abs(dQ[0].cpu().numpy()[rows, heads] - dq_ref).max() <= 2e-2
    krows = rng.integers(0, w.seq_total, 48)
    kheads = rng.integers(0, w.heads_kv, 48).astype(np.int32)
    dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, w.causal, pos, krows, kheads)
    assert np.abs(dK[0].cpu().numpy()[krows, kheads] - dk_ref).max() <= 2e-2
    assert np.abs(dV[0].cpu().numpy()[krows, kheads] - dv_ref).max() <= 2e-2


def test_rank_calls_refuse_lanes():
    from paper_2512_20968_b200 import binding as B
    from paper_2512_20968_b200 import plan_for

    w = W.scaled_down(W.C2, 128, heads_q=4, heads_kv=4)
    plan = plan_for(w, usp_lanes=2)
    x = torch.zeros(16, device="cuda")
    with pytest.raises(B.MeshAttnError) as e:
        plan.rank_fwd(0, x, x, x, x, x)
    assert e.value.status == B.EUNSUPPORTED
