"""GPU parity: mesh_attn_bwd_preprocess + mesh_attn_tile_bwd (through the C ABI) against the fp64
oracle on the same seeded bf16 inputs.  Tolerance (BASELINE.json): gradients within 2e-2 max abs."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.util import bits_to_f64, torch_bits

pytestmark = pytest.mark.gpu

TOL_GRAD = 2e-2


def run_fwd_bwd(w, inp, **overrides):
    from paper_2512_20968_b200 import Buffers, plan_for

    plan = plan_for(w, **overrides)
    buf = Buffers(plan, w, backward=True)
    plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
    for t in (buf.dQ, buf.dK, buf.dV):
        t.fill_(float("nan"))                     # mesh_attn_backward zeroes the accumulators itself
    plan.backward(inp["q"], inp["k"], inp["v"], buf.O, inp["do"], buf.lse, buf.bwd_ws, buf.dQ, buf.dK, buf.dV)
    torch.cuda.synchronize()
    return plan, buf


def check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads, qs_rows=None, bi=0, tol=TOL_GRAD):
    q, k, v, do = (torch_bits(inp[x][bi]) for x in ("q", "k", "v", "do"))
    pos = oracle.positions(w.n, w.L, w.seq_layout)
    dq_ref, _, delta_ref = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, qrows, qheads)
    dq = buf.dQ[bi].cpu().numpy()[qrows, qheads].astype(np.float64)
    delta = buf.delta[bi].cpu().numpy()[qheads, qrows].astype(np.float64)
    dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, w.causal, pos, krows, kheads, qs_rows=qs_rows)
    dk = buf.dK[bi].cpu().numpy()[krows, kheads].astype(np.float64)
    dv = buf.dV[bi].cpu().numpy()[krows, kheads].astype(np.float64)
    errs = dict(dq=np.abs(dq - dq_ref).max(), dk=np.abs(dk - dk_ref).max(), dv=np.abs(dv - dv_ref).max(),
                delta=np.abs(delta - delta_ref).max())
    assert np.isfinite(dq).all() and np.isfinite(dk).all() and np.isfinite(dv).all()
    # delta = dO . O inherits the forward's output error: |d delta| <= sum_d |dO_d| |dO_d err| ~ sqrt(D) * max|dO| ~ 5e-2
    assert errs["delta"] <= 5e-2, errs
    assert max(errs["dq"], errs["dk"], errs["dv"]) <= tol, errs
    return errs


def check_invariants(w, inp, buf, bi=0):
    """hold for any mask, per KV head: sum_t dV[t] = sum_s dO[s] (rows of P sum to 1), sum_t dK[t] = 0
    (rows of dS sum to 0), <Q,dQ> = <K,dK>."""
    g = w.heads_q // w.heads_kv
    do = inp["do"][bi].double()
    dV, dK, dQ = buf.dV[bi].double(), buf.dK[bi].double(), buf.dQ[bi].double()
    N = w.seq_total
    sum_do = do.view(N, w.heads_kv, g, w.head_dim).sum((0, 2))
    # N terms of per-element error <= 2e-2 add up like sqrt(N); outlier data adds a relative part (bf16 operands)
    tol = 2e-2 * max(1.0, N ** 0.5 / 8)
    assert (dV.sum(0) - sum_do).abs().max().item() <= tol + 4e-3 * sum_do.abs().max().item()
    assert dK.sum(0).abs().max().item() <= tol + 4e-3 * dK.abs().sum(0).max().item() / N ** 0.5
    a = (inp["q"][bi].double() * dQ).sum().item()
    b = (inp["k"][bi].double() * dK).sum().item()
    scale = (inp["q"][bi].double() * dQ).abs().sum().item()
    assert abs(a - b) <= 1e-3 * scale


def all_pairs(rows, heads):
    return np.repeat(np.asarray(rows, dtype=np.int64), len(heads)), np.tile(np.asarray(heads, dtype=np.int32), len(rows))


@pytest.mark.parametrize("name,L,hq", [("C2", 384, 4), ("C4", 128, 8)])
def test_scaled_configs_full_keys(oracle, name, L, hq):
    w = W.scaled_down(W.CONFIGS[name], L, heads_q=hq)
    inp = W.make_inputs(w, "cuda")
    _, buf = run_fwd_bwd(w, inp)
    rng = np.random.default_rng(3)
    rows = np.unique(np.concatenate([rng.integers(0, w.seq_total, 48), [0, w.seq_total - 1, w.L - 1, w.L]]))
    qrows, qheads = all_pairs(rows, [0, w.heads_q - 1])
    krows, kheads = all_pairs(rows[:24], [0, w.heads_kv - 1] if w.seq_total <= 4096 else [w.heads_kv - 1])
    check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
    check_invariants(w, inp, buf)


@pytest.mark.parametrize("name", ["C2", "C5"])
def test_paired_and_unpaired_kernel_variants(oracle, name):
    """The three tile_bwd kernels a pairable plan can run (plan desc field bwd_pairing): 2-CTA clusters with multicast Q / dO
    tiles AND the pair's dQ exchange (0 = auto, MESH_ATTN_Q_BWD_PAIRED == 2), single CTAs (1), clusters without the exchange (2):
    each against the oracle, and against each other (the exchange rounds half of the dQ partial sums to bf16)."""
    from paper_2512_20968_b200.binding import Q_BWD_PAIRED

    w = W.scaled_down(W.CONFIGS[name], 256, heads_q=2)
    if w.n > 16:
        w = replace(w, a=4, b=4, seq_total=16 * 256)         # C5's mask, layout and order on a 4 x 4 mesh
    inp = W.make_inputs(w, "cuda")
    rng = np.random.default_rng(5)
    rows = np.unique(np.concatenate([rng.integers(0, w.seq_total, 32), [0, w.seq_total - 1, w.L - 1, w.L]]))
    qrows, qheads = all_pairs(rows, range(w.heads_q))
    krows, kheads = all_pairs(rows[:16], range(w.heads_kv))
    bufs, errs = [], {}
    for pairing, mode in ((0, 2), (1, 0), (2, 1)):
        plan, buf = run_fwd_bwd(w, inp, bwd_pairing=pairing)
        assert plan.query(Q_BWD_PAIRED) == mode
        errs[mode] = check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
        check_invariants(w, inp, buf)
        plan.health()
        bufs.append(buf)
    print(f"\n{w.name} tile_bwd variants (2 = pair + dQ exchange, 0 = single CTA, 1 = pair): " + str({k: {a: float(f'{b:.3g}') for a, b in v.items()} for k, v in errs.items()}))
    for other in bufs[1:]:
        for x, y in ((bufs[0].dQ, other.dQ), (bufs[0].dK, other.dK), (bufs[0].dV, other.dV)):
            assert (x - y).abs().max().item() <= (1e-2 if x is bufs[0].dQ else 1e-3)   # atomics: the summation order is run-dependent; dQ: + the exchange's bf16 rounding
    with pytest.raises(Exception):
        run_fwd_bwd(w, inp, bwd_pairing=3)


def test_exchange_every_row_and_odd_paths(oracle):
    """The dQ exchange on EVERY query row and key of a small problem, for the three kinds of pairable plans: non-causal
    (items 2k, 2k+1 = neighbouring key blocks of one KV partition), striped causal (the same key block of two KV partitions,
    offsets 0 / -1), GQA (the Q walk repeats per query head of the group); and a non-pairable plan (contiguous causal) still
    runs the single-CTA kernel."""
    from paper_2512_20968_b200.binding import Q_BWD_PAIRED

    cases = [
        replace(W.scaled_down(W.C2, 256, heads_q=2), a=2, b=2, seq_total=4 * 256),
        replace(W.scaled_down(W.C4, 256, heads_q=4), a=2, b=2, seq_total=4 * 256, heads_kv=2),
        replace(W.scaled_down(W.C5, 512, heads_q=1), a=2, b=2, seq_total=4 * 512),
    ]
    for w in cases:
        inp = W.make_inputs(w, "cuda")
        plan, buf = run_fwd_bwd(w, inp)
        assert plan.query(Q_BWD_PAIRED) == 2
        qrows, qheads = all_pairs(np.arange(w.seq_total), range(w.heads_q))
        krows, kheads = all_pairs(np.arange(0, w.seq_total, 7), range(w.heads_kv))
        check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
        check_invariants(w, inp, buf)
    w = replace(cases[1], seq_layout="contiguous")
    inp = W.make_inputs(w, "cuda")
    plan, buf = run_fwd_bwd(w, inp)
    assert plan.query(Q_BWD_PAIRED) == 0
    check_grads(oracle, w, inp, buf, *all_pairs(np.arange(0, w.seq_total, 3), range(w.heads_q)), *all_pairs(np.arange(0, w.seq_total, 7), range(w.heads_kv)))


@pytest.mark.parametrize("pairing", [0, 1])
def test_sweep_pieces(oracle, pairing):
    """tile_bwd work items as (key block, piece of the Q sweep) (plan desc field bwd_piece_blocks): pieces of one segment, of two
    blocks' worth and the whole sweep give the same gradients (the same sums in another order), each within tolerance of the
    oracle on every row and key -- striped causal (pieces that end before a key block are pruned from the list), contiguous
    causal (they stay, as zero-step items), GQA, two Q chunks in greedy order."""
    from paper_2512_20968_b200.binding import Q_BWD_ITEMS_PER_GPU

    for layout in ("striped", "contiguous"):
        w = replace(W.scaled_down(W.C4, 512, heads_q=4), a=3, b=2, seq_total=6 * 512, heads_kv=2, seq_layout=layout, order="greedy", k_q=2, k_kv=2)
        inp = W.make_inputs(w, "cuda")
        qrows, qheads = all_pairs(np.arange(0, w.seq_total, 3), range(w.heads_q))
        krows, kheads = all_pairs(np.arange(0, w.seq_total, 5), range(w.heads_kv))
        ref, counts = None, []
        for blocks in (1, 4, 1 << 20):
            plan, buf = run_fwd_bwd(w, inp, bwd_piece_blocks=blocks, bwd_pairing=pairing)
            counts.append(plan.query(Q_BWD_ITEMS_PER_GPU))
            check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
            check_invariants(w, inp, buf)
            if ref is None:
                ref = buf
            else:
                for x, y in ((ref.dQ, buf.dQ), (ref.dK, buf.dK), (ref.dV, buf.dV)):
                    assert (x - y).abs().max().item() <= 1e-2
        assert counts[0] > counts[1] > counts[2]


@pytest.mark.parametrize("layout,kvr", [("contiguous", True), ("striped", False), ("striped", True)])
def test_causal_small_full(oracle, layout, kvr):
    """every row / key of a small causal problem (3x2 mesh, GQA 2:1): exercises diagonal blocks, fully masked
    pairs (contiguous), both tilings."""
    w = replace(W.scaled_down(W.C4, 128, heads_q=4), a=3, b=2, seq_total=6 * 128, heads_kv=2, seq_layout=layout, kvr=kvr)
    inp = W.make_inputs(w, "cuda")
    _, buf = run_fwd_bwd(w, inp)
    qrows, qheads = all_pairs(np.arange(w.seq_total), range(w.heads_q))
    krows, kheads = all_pairs(np.arange(w.seq_total), range(w.heads_kv))
    check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
    check_invariants(w, inp, buf)


def test_c5_shape_sparse_do_probe(oracle):
    """16x16 mesh, causal striped, greedy order, k_q = k_kv = 2 (configs[4] structure) at L = 256.
    dK/dV are checked in full-tensor fashion with the sparse-dO probe: dO non-zero on R sampled query rows
    only, so all of dK, dV depends on R oracle rows (gradients are linear in dO)."""
    w = W.scaled_down(W.C5, 256, heads_q=2)
    inp = W.make_inputs(w, "cuda")
    rng = np.random.default_rng(11)
    live = np.unique(np.concatenate([rng.integers(0, w.seq_total, 40), [w.seq_total - 1, 5 * w.L]]))
    mask = torch.zeros(w.seq_total, dtype=torch.bool, device="cuda")
    mask[torch.as_tensor(live, device="cuda")] = True
    inp["do"] = inp["do"] * mask[None, :, None, None]
    _, buf = run_fwd_bwd(w, inp)
    qrows, qheads = all_pairs(live, [0, 1])
    krows = np.unique(np.concatenate([rng.integers(0, w.seq_total, 200), [0, 1, w.L - 1, w.L, w.seq_total - 1]]))
    krows, kheads = all_pairs(krows, [0, 1])
    check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads, qs_rows=live)
    check_invariants(w, inp, buf)
    # rows with dO = 0 have dQ = 0 exactly
    assert torch.all(buf.dQ[0][~mask] == 0)


def test_batch_and_bhnd_layout(oracle):
    from paper_2512_20968_b200 import Buffers, plan_for

    w = replace(W.scaled_down(W.C4, 128, heads_q=4), batch=2, a=2, b=2, seq_total=4 * 128)
    inp = W.make_inputs(w, "cuda")
    _, buf = run_fwd_bwd(w, inp)
    rows = np.arange(0, w.seq_total, 7)
    for bi in range(2):
        qrows, qheads = all_pairs(rows, range(w.heads_q))
        krows, kheads = all_pairs(rows, range(w.heads_kv))
        check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads, bi=bi)
    inp_t = {kk: vv.permute(0, 2, 1, 3).contiguous() for kk, vv in inp.items()}
    plan = plan_for(w, tensor_layout=1)
    b2 = Buffers(plan, w, backward=True)
    tr = lambda t: torch.empty_like(t.permute(0, 2, 1, 3).contiguous())
    O_t, dQ_t, dK_t, dV_t = tr(b2.O), tr(b2.dQ), tr(b2.dK), tr(b2.dV)
    plan.forward(inp_t["q"], inp_t["k"], inp_t["v"], O_t, b2.lse, b2.partial_O, b2.partial_lse)
    plan.backward(inp_t["q"], inp_t["k"], inp_t["v"], O_t, inp_t["do"], b2.lse, b2.bwd_ws, dQ_t, dK_t, dV_t)
    torch.cuda.synchronize()
    # atomics make the summation order run-dependent: compare to tolerance, not bit-exactly
    for a, b in ((dQ_t, buf.dQ), (dK_t, buf.dK), (dV_t, buf.dV)):
        assert (a.permute(0, 2, 1, 3) - b).abs().max().item() <= 1e-3


def test_outlier_scores_c3_shape(oracle):
    """configs[2] structure: 4 of 128 Q/K channels x8 (|scaled score| up to ~100, |dK| up to ~100), causal striped 4x4,
    greedy order.  The 2e-2 absolute bar is a ~2e-4 relative bar on this data, below the 2^-9 rounding of a single bf16
    MMA operand: plan precision = 1 (P and dS split into hi + lo bf16 operands) is the mode that has to meet it
    (DESIGN.md "precision"); the single-operand mode is run too and its error reported."""
    w = W.scaled_down(W.C3, 512, heads_q=2)
    inp = W.make_inputs(w, "cuda")
    rng = np.random.default_rng(5)
    rows = np.unique(rng.integers(0, w.seq_total, 48))
    qrows, qheads = all_pairs(rows, [0, 1])
    krows, kheads = all_pairs(rows[:24], [0, 1])
    _, buf = run_fwd_bwd(w, inp, precision=0)
    errs = check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads, tol=0.5)
    print("C3-shape single-bf16 operand errors:", errs)
    _, buf = run_fwd_bwd(w, inp, precision=1)
    errs = check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads, tol=TOL_GRAD)
    print("C3-shape split (hi+lo) operand errors:", errs)
    check_invariants(w, inp, buf)


def test_split_precision_iid(oracle):
    """precision = 1 on iid data (GQA, causal, both layouts of the work list exercised by C4's structure)."""
    w = W.scaled_down(W.C4, 256, heads_q=8)
    inp = W.make_inputs(w, "cuda")
    _, buf = run_fwd_bwd(w, inp, precision=1)
    rng = np.random.default_rng(9)
    rows = np.unique(np.concatenate([rng.integers(0, w.seq_total, 40), [0, w.seq_total - 1]]))
    qrows, qheads = all_pairs(rows, [0, w.heads_q - 1])
    krows, kheads = all_pairs(rows[:20], [0, w.heads_kv - 1])
    errs = check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
    assert max(errs["dq"], errs["dk"], errs["dv"]) <= 5e-3, errs     # an order of magnitude inside the bar
    check_invariants(w, inp, buf)


@pytest.mark.parametrize("batch,lanes", [(1, 1), (1, 2), (2, 1)])
def test_step_host_matches_device_calls_and_profile_counters(batch, lanes):
    """mesh_attn_step_host (host buffers; H2D, forward, backward and D2H overlapped on its copy streams: when batch == 1, Q up
    and dQ down per Q group, K, V up and dK, dV down per KV column around the first forward wave / last backward group, which
    then run one launch per simulated GPU; whole tensors otherwise) gives what the device-pointer calls give, twice in a row;
    the per-kernel event profile counts one record per launch."""
    from paper_2512_20968_b200 import Buffers
    from paper_2512_20968_b200 import binding as B

    w = replace(W.scaled_down(W.C4, 256, heads_q=4), a=2, b=3, seq_total=6 * 256, heads_kv=2, batch=batch)
    inp = W.make_inputs(w, "cuda")
    plan, ref = run_fwd_bwd(w, inp, usp_lanes=lanes)
    host_in = {k: v.cpu().pin_memory() for k, v in inp.items()}
    buf = Buffers(plan, w, backward=True)
    dev = {k: torch.empty_like(v) for k, v in inp.items()}
    out = {k: torch.empty(t.shape, dtype=t.dtype).pin_memory() for k, t in
           dict(O=buf.O, lse=buf.lse, dQ=buf.dQ, dK=buf.dK, dV=buf.dV).items()}
    for rep in range(2):
        for t in list(dev.values()) + [buf.O, buf.lse, buf.dQ, buf.dK, buf.dV]:
            t.fill_(float("nan")) if t.is_floating_point() else t.zero_()
        for t in out.values():
            t.fill_(float("nan"))
        torch.cuda.synchronize()
        B.profile_enable(True, 64)
        plan.step_host(Q_host=host_in["q"], K_host=host_in["k"], V_host=host_in["v"], dO_host=host_in["do"],
                       O_host=out["O"], lse_host=out["lse"], dQ_host=out["dQ"], dK_host=out["dK"], dV_host=out["dV"],
                       d_Q=dev["q"], d_K=dev["k"], d_V=dev["v"], d_dO=dev["do"], d_O=buf.O, d_lse=buf.lse, d_bwd_ws=buf.bwd_ws,
                       d_dQ=buf.dQ, d_dK=buf.dK, d_dV=buf.dV, d_partial_O=buf.partial_O, d_partial_lse=buf.partial_lse)
        counts = {k: B.profile_read(k)[1] for k in (B.K_TILE_FWD, B.K_MERGE, B.K_BWD_PREPROCESS, B.K_TILE_BWD)}
        B.profile_enable(False)
        waves = w.b * lanes
        tiles = waves + (w.a - 1 if batch == 1 else 0)      # one wave / group split into its a simulated GPUs
        assert counts == {B.K_TILE_FWD: tiles, B.K_MERGE: waves, B.K_BWD_PREPROCESS: 1, B.K_TILE_BWD: tiles}
        assert torch.equal(out["O"], ref.O.cpu()) and torch.equal(out["lse"], ref.lse.cpu())   # forward is deterministic
        for name, t in (("dQ", ref.dQ), ("dK", ref.dK), ("dV", ref.dV)):                      # atomics: order-dependent last bits
            assert (out[name] - t.cpu()).abs().max().item() <= 1e-3


@pytest.mark.parametrize("kvr,a,b", [(False, 3, 2), (True, 4, 1), (False, 1, 4)])
def test_step_host_kv_columns_of_other_footprints(kvr, a, b):
    """The per-column copies of mesh_attn_step_host follow I^KV: contiguous footprints (no rotation), a mesh with
    a > b, one Q group only (b = 1: the first wave is also the last group), and a = 1 (no columns: whole K, V, dK, dV).
    Staging and host outputs start as NaN, so a partition that was not copied, or copied before it was final, shows."""
    from paper_2512_20968_b200 import Buffers

    w = replace(W.scaled_down(W.C4, 256, heads_q=4), a=a, b=b, seq_total=a * b * 256, heads_kv=2, kvr=kvr)
    inp = W.make_inputs(w, "cuda")
    plan, ref = run_fwd_bwd(w, inp)
    host_in = {k: v.cpu().pin_memory() for k, v in inp.items()}
    buf = Buffers(plan, w, backward=True)
    dev = {k: torch.empty_like(v) for k, v in inp.items()}
    for t in dev.values():
        t.view(torch.int16).fill_(0x7FC0)
    for t in (buf.O, buf.lse, buf.dQ, buf.dK, buf.dV):
        t.fill_(float("nan"))
    out = {k: torch.full(t.shape, float("nan"), dtype=t.dtype).pin_memory() for k, t in
           dict(O=buf.O, lse=buf.lse, dQ=buf.dQ, dK=buf.dK, dV=buf.dV).items()}
    plan.step_host(Q_host=host_in["q"], K_host=host_in["k"], V_host=host_in["v"], dO_host=host_in["do"],
                   O_host=out["O"], lse_host=out["lse"], dQ_host=out["dQ"], dK_host=out["dK"], dV_host=out["dV"],
                   d_Q=dev["q"], d_K=dev["k"], d_V=dev["v"], d_dO=dev["do"], d_O=buf.O, d_lse=buf.lse, d_bwd_ws=buf.bwd_ws,
                   d_dQ=buf.dQ, d_dK=buf.dK, d_dV=buf.dV, d_partial_O=buf.partial_O, d_partial_lse=buf.partial_lse)
    plan.health()
    for k in ("q", "k", "v", "do"):
        assert torch.equal(dev[k].view(torch.int16), inp[k].view(torch.int16)), k
    assert torch.equal(out["O"], ref.O.cpu()) and torch.equal(out["lse"], ref.lse.cpu())
    for name, t in (("dQ", ref.dQ), ("dK", ref.dK), ("dV", ref.dV)):
        assert torch.isfinite(out[name]).all(), name
        assert (out[name] - t.cpu()).abs().max().item() <= 1e-3, name
        assert torch.equal(out[name], getattr(buf, name).cpu()), name        # what came down is what the device holds at the end


@pytest.mark.parametrize("causal", [False, True])
def test_head_dim_64(oracle, causal):
    """head_dim 64 (BASELINE.json configs[0]'s heads) through the backward: the head_dim-128 kernel on tiles whose upper
    64 columns the TMA zero-fills; every row and key of a 2 x 2 mesh, both kernel variants (4 / 6 items per GPU pair up,
    the contiguous causal layout does not)."""
    w = replace(W.scaled_down(W.C1, 256), backward=True, causal=causal, seq_layout="striped" if causal else "contiguous")
    assert w.head_dim == 64
    inp = W.make_inputs(w, "cuda")
    _, buf = run_fwd_bwd(w, inp)
    qrows, qheads = all_pairs(np.arange(w.seq_total), range(w.heads_q))
    krows, kheads = all_pairs(np.arange(w.seq_total), range(w.heads_kv))
    check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads)
    check_invariants(w, inp, buf)
    if causal:
        w2 = replace(w, seq_layout="contiguous")
        _, buf2 = run_fwd_bwd(w2, inp)
        check_grads(oracle, w2, inp, buf2, qrows, qheads, krows, kheads)
