"""Plan desc field out_dtype = 1 (include/mesh_attn.h): O, dQ, dK, dV as bf16 -- an option of the boundary beyond the paper
("unpinned": SURVEY.md 8(b)).  Checked against the fp32 path of the same kernels and against the fp64 oracle:

  * forward: O (bf16) is EXACTLY the fp32 path's O rounded to nearest even (the merge rounds its fp32 sum once), lse is identical;
  * backward: the preprocess reads the bf16 O, the atomics accumulate in fp32 behind the planes of bwd_ws, three cast launches
    round the sums.  dV does not depend on O: bf16 resolution (2^-8 relative) of the fp32 path's values.  dQ and dK do, through
    delta = rowsum(dO o O): |d delta| <= 2^-9 sum_d |dO_d O_d|, up to ~1e-1 on rows that see few keys (|O| ~ |V|), which reaches
    dQ, dK times P K scale -- measured 1.6e-2 on the causal case; the bound used is 2 x the gradient tolerance (4e-2);
  * mesh_attn_step_host moves half the output bytes and returns the same tensors; forward_static follows the field too;
  * backward_goo and the per-rank calls refuse such a plan (EUNSUPPORTED); MESH_ATTN_Q_BWD_WS_BYTES grows by the accumulators."""
import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.test_gpu_backward import TOL_GRAD, all_pairs, run_fwd_bwd
from tests.util import torch_bits

pytestmark = pytest.mark.gpu

BF16_REL = 2.0 ** -8         # one bf16 rounding (2^-9) of the output + one of O inside delta, with margin


def _close_bf16(got, ref, what, abs_tol=TOL_GRAD * 0.25):
    got, ref = got.double(), ref.double()
    err = (got - ref).abs()
    bound = abs_tol + BF16_REL * ref.abs()
    assert torch.isfinite(got).all(), what
    assert (err <= bound).all(), f"{what}: max excess {(err - bound).max().item():.3e}, max err {err.max().item():.3e}"
    return err.max().item()


@pytest.mark.parametrize("causal,hd", [(True, 128), (False, 128), (False, 64)])
def test_bf16_outputs_match_fp32_path_and_oracle(oracle, causal, hd):
    import paper_2512_20968_b200.binding as B

    w = W.Workload("bf16out", 31, causal, 2, 2, 1, 2048, 4, 2, hd, seq_layout="striped" if causal else "contiguous")
    inp = W.make_inputs(w, "cuda")
    p32, b32 = run_fwd_bwd(w, inp)
    p16, b16 = run_fwd_bwd(w, inp, out_dtype=1)
    p16.health()
    assert b16.O.dtype == torch.bfloat16 and b16.dQ.dtype == torch.bfloat16
    acc_bytes = w.batch * w.seq_total * (w.heads_q + 2 * w.heads_kv) * w.head_dim * 4
    assert p16.query(B.Q_BWD_WS_BYTES) == p32.query(B.Q_BWD_WS_BYTES) + acc_bytes

    # forward: one rounding of the same fp32 sum
    assert torch.equal(b16.lse, b32.lse)
    assert torch.equal(b16.O, b32.O.to(torch.bfloat16))
    # backward against the fp32 path
    errs = {n: _close_bf16(getattr(b16, n), getattr(b32, n), n, abs_tol=TOL_GRAD * (0.25 if n == "dV" else 2.0)) for n in ("dQ", "dK", "dV")}
    # ... and against the oracle on sampled rows / keys of every partition
    rng = np.random.default_rng(31)
    rows = np.unique(np.concatenate([[p * w.L, p * w.L + w.L - 1] + list(p * w.L + rng.integers(0, w.L, 6)) for p in range(w.n)]))
    qr, qh = all_pairs(rows, list(range(w.heads_q)))
    kr, kh = all_pairs(rows, list(range(w.heads_kv)))
    q, k, v, do = (torch_bits(inp[x][0]) for x in ("q", "k", "v", "do"))
    pos = oracle.positions(w.n, w.L, w.seq_layout)
    O_ref, _ = oracle.fwd_rows(q, k, v, w.scale, w.causal, pos, qr, qh)
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, qr, qh)
    dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, w.causal, pos, kr, kh)
    for name, got, ref in (("O", b16.O[0].float().cpu().numpy()[qr, qh], O_ref), ("dQ", b16.dQ[0].float().cpu().numpy()[qr, qh], dq_ref),
                           ("dK", b16.dK[0].float().cpu().numpy()[kr, kh], dk_ref), ("dV", b16.dV[0].float().cpu().numpy()[kr, kh], dv_ref)):
        err = np.abs(got.astype(np.float64) - ref)
        bound = {"O": 1e-2, "dV": TOL_GRAD}.get(name, 2 * TOL_GRAD) + BF16_REL * np.abs(ref)
        assert (err <= bound).all(), (name, err.max())
        errs[name + "_oracle"] = err.max()
    print(f"\nout_dtype=1 causal={causal} head_dim={hd}: " + ", ".join(f"{k_}={v_:.2e}" for k_, v_ in errs.items()))

    # forward_static follows the field
    need, cap = p16.forward_static_limits()
    assert need <= cap
    O_s, lse_s = torch.full_like(b16.O, float("nan")), torch.full_like(b16.lse, float("nan"))
    p16.forward_static(inp["q"], inp["k"], inp["v"], O_s, lse_s)
    torch.cuda.synchronize()
    assert torch.equal(O_s, b16.O) and torch.equal(lse_s, b16.lse)

    # calls that accumulate into caller-owned fp32 gradients refuse the plan
    with pytest.raises(B.MeshAttnError) as e:
        p16.backward_goo(0, inp["q"], inp["k"], inp["v"], inp["do"], b16.bwd_ws, b32.dQ, b32.dK, b32.dV)
    assert e.value.status == -2


@pytest.mark.parametrize("batch,layout", [(1, 0), (2, 0), (1, 1)])
def test_step_host_bf16_outputs(batch, layout):
    """mesh_attn_step_host with out_dtype = 1: by Q group (batch 1, [B,N,H,D]) and whole-tensor copies; the host tensors equal
    the device calls' results (forward exactly; gradients up to the order of the fp32 atomics, then one rounding)."""
    from paper_2512_20968_b200 import Buffers, plan_for

    w = W.Workload("bf16host", 32, True, 2, 2, batch, 2048, 4, 2, 128, seq_layout="striped")
    inp = W.make_inputs(w, "cuda")
    if layout == 1:
        inp = {k_: v_.permute(0, 2, 1, 3).contiguous() for k_, v_ in inp.items()}
    plan = plan_for(w, out_dtype=1, tensor_layout=layout)
    ref = Buffers(plan, w, backward=True)
    if layout == 1:
        for n in ("O", "dQ", "dK", "dV"):
            setattr(ref, n, getattr(ref, n).permute(0, 2, 1, 3).contiguous())
    plan.forward(inp["q"], inp["k"], inp["v"], ref.O, ref.lse, ref.partial_O, ref.partial_lse)
    plan.backward(inp["q"], inp["k"], inp["v"], ref.O, inp["do"], ref.lse, ref.bwd_ws, ref.dQ, ref.dK, ref.dV)
    torch.cuda.synchronize()

    host_in = {k_: v_.cpu().pin_memory() for k_, v_ in inp.items()}
    buf = Buffers(plan, w, backward=True)
    dev = {k_: torch.empty_like(v_) for k_, v_ in inp.items()}
    outs = dict(O=ref.O, lse=ref.lse, dQ=ref.dQ, dK=ref.dK, dV=ref.dV)
    out = {k_: torch.empty(t.shape, dtype=t.dtype).pin_memory() for k_, t in outs.items()}
    dbuf = {k_: torch.full_like(t, float("nan")) for k_, t in outs.items()}
    for t in list(dev.values()):
        t.view(torch.int16).fill_(0x7FC0)                  # NaN bits: a copy that did not happen shows
    for t in out.values():
        t.fill_(float("nan"))
    plan.step_host(Q_host=host_in["q"], K_host=host_in["k"], V_host=host_in["v"], dO_host=host_in["do"],
                   O_host=out["O"], lse_host=out["lse"], dQ_host=out["dQ"], dK_host=out["dK"], dV_host=out["dV"],
                   d_Q=dev["q"], d_K=dev["k"], d_V=dev["v"], d_dO=dev["do"], d_O=dbuf["O"], d_lse=dbuf["lse"], d_bwd_ws=buf.bwd_ws,
                   d_dQ=dbuf["dQ"], d_dK=dbuf["dK"], d_dV=dbuf["dV"], d_partial_O=buf.partial_O, d_partial_lse=buf.partial_lse)
    plan.health()
    assert out["O"].dtype == torch.bfloat16 and torch.equal(out["O"], ref.O.cpu()) and torch.equal(out["lse"], ref.lse.cpu())
    for n in ("dQ", "dK", "dV"):
        got, want = out[n].double(), outs[n].cpu().double()
        assert torch.isfinite(got).all(), n
        assert ((got - want).abs() <= 1e-3 + 2.0 ** -7 * want.abs()).all(), n        # atomics order, then at most one bf16 ulp apart
