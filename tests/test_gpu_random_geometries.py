"""GPU parity on RANDOM plan geometries: seeded draws over mesh shape (a x b, also a != b and a or b = 1), partition length
(1..5 key blocks, so ragged against the 256-row forward items and the backward's pairing), heads / GQA group, head_dim,
outlier data with the hi+lo operand mode, mask and sequence layout, KV rotation, tile order with k_Q x k_KV chunks, batch, Mesh-USP lanes and the kernel-variant fields
(bwd_piece_blocks, bwd_pairing, fwd_pairing) -- the combinations the named BASELINE.json shapes do not reach.  Every draw runs mesh_attn_forward + mesh_attn_backward through the C ABI and is
compared with the fp64 oracle (forward: sampled rows of every partition incl. its first and last row, all heads; backward:
sampled query rows and keys, plus the three gradient invariants), tolerances of BASELINE.json.  The draw list is fixed by
the seeds below; `geometry(seed)` is also exercised on the CPU (tests/test_planner.py) so that an invalid draw shows there."""
import os
from dataclasses import replace

import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W

SEEDS = list(range(int(os.environ.get("MESH_ATTN_TEST_DRAWS", "20"))))     # a longer hunt: MESH_ATTN_TEST_DRAWS=300 python -m pytest tests/test_gpu_random_geometries.py -m gpu


def geometry(seed):
    """-> (Workload, plan overrides).  Pure host arithmetic: callable without a GPU."""
    rng = np.random.default_rng(9000 + seed)
    while True:
        a, b = int(rng.integers(1, 5)), int(rng.integers(1, 5))
        if a * b <= 12:
            break
    k_q, k_kv = (int(rng.choice([1, 2])), int(rng.choice([1, 2])))
    blocks = int(rng.integers(1, 6))                                     # 128-row blocks per partition
    L = 128 * blocks * max(k_q, k_kv) if rng.random() < 0.5 else 128 * blocks
    if L % (128 * k_q) or L % (128 * k_kv):
        k_q = k_kv = 1
    heads_kv = int(rng.choice([1, 2]))
    group = int(rng.choice([1, 2, 4]))
    causal = bool(rng.random() < 0.6)
    lanes = 2 if heads_kv == 2 and rng.random() < 0.7 else 1
    w = W.Workload(name=f"rand{seed}", index=100 + seed, causal=causal, a=a, b=b, batch=int(rng.choice([1, 1, 2])),
                   seq_total=a * b * L, heads_q=heads_kv * group, heads_kv=heads_kv, head_dim=int(rng.choice([64, 128, 128])),
                   kvr=bool(rng.random() < 0.6), order="greedy" if rng.random() < 0.5 else "row_major", k_q=k_q, k_kv=k_kv,
                   seq_layout="striped" if causal and rng.random() < 0.6 else "contiguous")
    if w.head_dim == 128 and rng.random() < 0.25:                         # C3's data: 4 Q / K channels x 8, run with hi+lo operands (precision 1)
        w = replace(w, outlier=True)
    # the kernel-variant fields of the plan desc: sweep pieces of the backward, the three backward kernels, the two forward kernels
    variants = dict(bwd_piece_blocks=int(rng.choice([0, 0, 1, 2, 3, 7])), bwd_pairing=int(rng.choice([0, 0, 0, 1, 2])),
                    fwd_pairing=int(rng.choice([0, 0, 1])), partial_mode=int(rng.choice([0, 0, 0, 1])))    # 1: per-pair partials
    return w, dict(usp_lanes=lanes, **variants)


@pytest.mark.gpu
@pytest.mark.parametrize("seed", SEEDS)
def test_random_geometry_against_oracle(oracle, seed):
    from tests.test_gpu_backward import all_pairs, check_grads, check_invariants, run_fwd_bwd
    from tests.test_gpu_forward import check_against_oracle

    w, overrides = geometry(seed)
    inp = W.make_inputs(w, "cuda")
    plan, buf = run_fwd_bwd(w, inp, **overrides)
    plan.health()
    rng = np.random.default_rng(9500 + seed)
    edge = np.concatenate([[p * w.L, p * w.L + w.L - 1] for p in range(w.n)])
    rows = np.unique(np.concatenate([edge, rng.integers(0, w.seq_total, 40)]))
    heads = list(range(w.heads_q))
    for bi in range(w.batch):
        fwd = check_against_oracle(oracle, w, inp, buf.O[bi].cpu().numpy(), buf.lse[bi].cpu().numpy(), rows=rows, heads=heads, batch_index=bi)
        qrows, qheads = all_pairs(rows, heads)
        krows, kheads = all_pairs(np.unique(np.concatenate([edge[:8], rng.integers(0, w.seq_total, 24)])), range(w.heads_kv))
        errs = check_grads(oracle, w, inp, buf, qrows, qheads, krows, kheads, bi=bi)
        check_invariants(w, inp, buf, bi=bi)
    print(f"\nseed {seed}: {w.a}x{w.b} L={w.L} B={w.batch} Hq/Hkv={w.heads_q}/{w.heads_kv} D={w.head_dim} causal={w.causal} {w.seq_layout} "
          f"kvr={w.kvr} {w.order} k={w.k_q}x{w.k_kv} lanes={overrides['usp_lanes']}: O {fwd[0]:.2e} lse {fwd[2]:.2e} "
          + " ".join(f"{k}={v:.2e}" for k, v in errs.items()))


@pytest.mark.gpu
@pytest.mark.parametrize("seed", SEEDS[::2])
def test_random_geometry_step_host(seed):
    """mesh_attn_step_host on the same draws (its copies are cut by Q group and KV column when batch == 1, whole tensors
    otherwise; USP lanes change which wave / group is first / last): NaN-filled staging and host outputs, result against the
    device-pointer calls (forward bit-identical; gradients up to the order of the fp32 atomics)."""
    from paper_2512_20968_b200 import Buffers
    from tests.test_gpu_backward import run_fwd_bwd

    w, overrides = geometry(seed)
    inp = W.make_inputs(w, "cuda")
    plan, ref = run_fwd_bwd(w, inp, **overrides)
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
        assert (out[name] - t.cpu()).abs().max().item() <= 1e-3 * max(1.0, t.abs().max().item()), name     # the order of the fp32 atomics differs run to run
        assert torch.equal(out[name], getattr(buf, name).cpu()), name


@pytest.mark.gpu
@pytest.mark.parametrize("seed", SEEDS[1::2])
def test_random_geometry_goo_executors(seed):
    """mesh_attn_forward_goo / mesh_attn_backward_goo (the step lists executed task by task, copies standing in for the
    collectives) on the other half of the draws, Q group by Q group of every lane, against the fused calls: O at the level of the
    bf16 P operand (each task rounds against its own running max), lse to 1e-4, gradients up to the order of the fp32 atomics."""
    from paper_2512_20968_b200 import binding as B
    from tests.test_gpu_backward import run_fwd_bwd

    w, overrides = geometry(seed)
    inp = W.make_inputs(w, "cuda")
    plan, ref = run_fwd_bwd(w, inp, **overrides)
    f32 = dict(dtype=torch.float32, device="cuda")
    part_O = torch.full((plan.query(B.Q_GOO_PARTIAL_O_BYTES) * w.a // 4,), float("nan"), **f32)
    part_lse = torch.full((plan.query(B.Q_GOO_PARTIAL_LSE_BYTES) * w.a // 4,), float("nan"), **f32)
    comm_ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    O, lse = torch.full_like(ref.O, float("nan")), torch.full_like(ref.lse, float("nan"))
    dQ, dK, dV = torch.zeros_like(ref.dQ), torch.zeros_like(ref.dK), torch.zeros_like(ref.dV)
    for r in range(w.b * overrides["usp_lanes"]):
        plan.forward_goo(r, inp["q"], inp["k"], inp["v"], O, lse, part_O, part_lse, comm_ws=comm_ws, comm_repeat=seed % 3, overlap=bool(seed % 4))
        plan.backward_goo(r, inp["q"], inp["k"], inp["v"], inp["do"], ref.bwd_ws, dQ, dK, dV, comm_ws=comm_ws, comm_repeat=seed % 3, overlap=bool(seed % 4))
    torch.cuda.synchronize()
    plan.health()
    # two evaluations that round P to bf16 against different running maxima (per task / per pair / fused): each is off by at most
    # 2^-9 sum_t p_t |v_t| <= 2^-9 max|V| per element (the rows that come close see two or three keys), so they are at most twice
    # that apart; each is within 1e-2 of the oracle (test_random_geometry_against_oracle).  Seen over 300 draws: up to 8.6e-3.
    assert (O - ref.O).abs().max().item() <= 2 * 2.0 ** -9 * inp["v"].float().abs().max().item()
    fin = torch.isfinite(ref.lse)
    assert torch.equal(torch.isfinite(lse), fin) and (lse[fin] - ref.lse[fin]).abs().max().item() <= 1e-4
    for name, got, want in (("dQ", dQ, ref.dQ), ("dK", dK, ref.dK), ("dV", dV, ref.dV)):
        assert torch.isfinite(got).all(), name
        err = (got - want).abs().max().item()
        # the fused backward's pair exchange rounds half of the dQ partial sums to bf16; the executor's single-CTA launches do not
        assert err <= (1e-2 if name == "dQ" else 1e-3) * max(1.0, want.abs().max().item()), f"{name}: {err:.3e} vs mesh_attn_backward"


def _rank_draws():
    out = []
    for seed in SEEDS:
        w, overrides = geometry(seed)
        if w.kvr and w.batch == 1 and overrides["usp_lanes"] == 1:      # the reduce-scatter of dK, dV needs g in I_g^KV (rotation)
            out.append(seed)
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("seed", _rank_draws())
def test_random_geometry_rank_calls(seed):
    """The per-rank calls (one GPU's share of Alg.2 / Alg.3 on its gathered partitions, the n ranks played one after the other,
    reduce-scatters through the peer-memory reducers) on the draws with KV rotation: forward bit-identical to the simulated-GPU
    path, gradients up to the order of the fp32 atomics (and the pair exchange's bf16 halves of dQ, which the per-rank backward,
    pairing inside its own lists, may group differently)."""
    from tests.test_gpu_backward import run_fwd_bwd
    from tests.test_gpu_rank_calls import play_ranks

    w, _ = geometry(seed)
    inp = W.make_inputs(w, "cuda")
    plan, ref = run_fwd_bwd(w, inp)
    O, lse, grads = play_ranks(plan, w, inp)
    plan.health()
    assert torch.equal(O, ref.O) and torch.equal(lse, ref.lse)
    for name, got, want in zip(("dQ", "dK", "dV"), grads, (ref.dQ, ref.dK, ref.dV)):
        assert torch.isfinite(got).all(), name
        err = (got - want).abs().max().item()
        assert err <= (1e-2 if name == "dQ" else 1e-3) * max(1.0, want.abs().max().item()), f"{name}: {err:.3e} vs the simulated-GPU path"


@pytest.mark.gpu
@pytest.mark.parametrize("seed", SEEDS[::3])
def test_random_geometry_bf16_outputs_and_static_forward(seed):
    """Plan desc field out_dtype = 1 and mesh_attn_forward_static on the draws: O (bf16) is the fp32 path's O rounded once, lse is
    identical, dV within bf16 resolution of the fp32 path's, dQ / dK within the error the rounded O leaves in delta
    (tests/test_gpu_out_dtype.py); the no-allocation forward returns the same bits wherever the plan fits its 32 MiB array."""
    from tests.test_gpu_backward import TOL_GRAD, run_fwd_bwd

    w, overrides = geometry(seed)
    inp = W.make_inputs(w, "cuda")
    _, b32 = run_fwd_bwd(w, inp, **overrides)
    p16, b16 = run_fwd_bwd(w, inp, out_dtype=1, **overrides)
    p16.health()
    assert torch.equal(b16.lse, b32.lse) and torch.equal(b16.O, b32.O.to(torch.bfloat16))
    for name, abs_tol in (("dQ", 2 * TOL_GRAD), ("dK", 2 * TOL_GRAD), ("dV", 0.25 * TOL_GRAD)):
        got, ref = getattr(b16, name).double(), getattr(b32, name).double()
        assert torch.isfinite(got).all(), name
        if w.outlier and name != "dV":       # |K|, |Q| x 8 multiply what the rounded O leaves in delta: outside the gradient bar by design
            continue                         # (out_dtype: outlier data keeps fp32 outputs)
        assert ((got - ref).abs() <= abs_tol + 2.0 ** -8 * ref.abs()).all(), name
    need, cap = p16.forward_static_limits()
    if need <= cap:
        O_s, lse_s = torch.full_like(b16.O, float("nan")), torch.full_like(b16.lse, float("nan"))
        p16.forward_static(inp["q"], inp["k"], inp["v"], O_s, lse_s)
        torch.cuda.synchronize()
        assert torch.equal(O_s, b16.O) and torch.equal(lse_s, b16.lse)
    print(f"\nseed {seed}: forward_static {'run' if need <= cap else 'refused'} ({need} of {cap} bytes)")


@pytest.mark.gpu
@pytest.mark.parametrize("seed", SEEDS[::4])
def test_random_geometry_bhnd_layout(seed):
    """tensor_layout = 1 ([B,H,N,D] tensors: other TMA maps, other strides in merge / preprocess / the dQ reduce boxes) on the draws:
    forward bit-identical to the [B,N,H,D] plan's, gradients up to the order of the fp32 atomics; mesh_attn_step_host in this layout
    (whole-tensor copies) returns the same tensors."""
    from paper_2512_20968_b200 import Buffers, plan_for
    from tests.test_gpu_backward import run_fwd_bwd

    w, overrides = geometry(seed)
    inp = W.make_inputs(w, "cuda")
    _, ref = run_fwd_bwd(w, inp, **overrides)
    tr = lambda t: t.permute(0, 2, 1, 3).contiguous()                      # noqa: E731
    inp_t = {k: tr(v) for k, v in inp.items()}
    plan = plan_for(w, tensor_layout=1, **overrides)
    buf = Buffers(plan, w, backward=True)
    O, dQ, dK, dV = (torch.full_like(tr(t), float("nan")) for t in (buf.O, buf.dQ, buf.dK, buf.dV))
    plan.forward(inp_t["q"], inp_t["k"], inp_t["v"], O, buf.lse, buf.partial_O, buf.partial_lse)
    plan.backward(inp_t["q"], inp_t["k"], inp_t["v"], O, inp_t["do"], buf.lse, buf.bwd_ws, dQ, dK, dV)
    torch.cuda.synchronize()
    plan.health()
    assert torch.equal(tr(O), ref.O) and torch.equal(buf.lse, ref.lse)
    for name, got, want in (("dQ", dQ, ref.dQ), ("dK", dK, ref.dK), ("dV", dV, ref.dV)):
        assert (tr(got) - want).abs().max().item() <= 1e-3 * max(1.0, want.abs().max().item()), name
    host_in = {k: v.cpu().pin_memory() for k, v in inp_t.items()}
    dev = {k: torch.full_like(v, float("nan")) for k, v in inp_t.items()}
    outs = dict(O=O, lse=buf.lse, dQ=dQ, dK=dK, dV=dV)
    out = {k: torch.full(t.shape, float("nan"), dtype=t.dtype).pin_memory() for k, t in outs.items()}
    dbuf = {k: torch.full_like(t, float("nan")) for k, t in outs.items()}
    plan.step_host(Q_host=host_in["q"], K_host=host_in["k"], V_host=host_in["v"], dO_host=host_in["do"],
                   O_host=out["O"], lse_host=out["lse"], dQ_host=out["dQ"], dK_host=out["dK"], dV_host=out["dV"],
                   d_Q=dev["q"], d_K=dev["k"], d_V=dev["v"], d_dO=dev["do"], d_O=dbuf["O"], d_lse=dbuf["lse"], d_bwd_ws=buf.bwd_ws,
                   d_dQ=dbuf["dQ"], d_dK=dbuf["dK"], d_dV=dbuf["dV"], d_partial_O=buf.partial_O, d_partial_lse=buf.partial_lse)
    plan.health()
    assert torch.equal(out["O"], O.cpu()) and torch.equal(out["lse"], buf.lse.cpu())
    for name in ("dQ", "dK", "dV"):
        want = outs[name].cpu()
        assert torch.isfinite(out[name]).all(), name
        assert (out[name] - want).abs().max().item() <= 1e-3 * max(1.0, want.abs().max().item()), name
