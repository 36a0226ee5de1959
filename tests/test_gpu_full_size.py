"""GPU parity at BASELINE.json's FULL sizes (configs[1..4]), in the launch configuration bench.py times
(mesh_attn_forward + mesh_attn_backward through the C ABI), on outputs the fp64 oracle can compute one by one:

  * O, LSE and dQ on sampled query rows of EVERY Q partition (first / last / random local rows): each row costs the
    oracle 4*N*D flops, and the sample touches every simulated GPU and every (Q_u, KV_v) pair;
  * causal configs: dK, dV of the keys at the last R token positions, which only the last R queries see -- exact with
    R oracle rows (under the striped layout they live in R different partitions);
  * non-causal config: dK, dV of sampled keys with the sparse-dO probe (dO non-zero on R query rows only; gradients are
    linear in dO, so ALL of dK, dV depends on R oracle rows);
  * properties that hold at any size: sum_t dV = sum_s dO, sum_t dK = 0, <Q,dQ> = <K,dK> (per KV head / globally).

Tolerances are BASELINE.json's.  configs[2] (outlier scores) runs with plan precision = 1."""
import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.util import torch_bits

pytestmark = pytest.mark.gpu

TOL_O_MAX, TOL_O_MEAN, TOL_LSE, TOL_GRAD = 1e-2, 1e-3, 1e-3, 2e-2
TAIL = 48          # causal: keys at the last TAIL positions


def _sub_bits(t, h0, h1):
    """[N, h1-h0, D] bf16 bits of heads h0..h1-1 of batch 0 on the host"""
    return torch_bits(t[0, :, h0:h1, :].contiguous())


def _invariants(w, inp, buf):
    g = w.heads_q // w.heads_kv
    N, chunk = w.seq_total, 1 << 16
    z = lambda: torch.zeros((w.heads_kv, w.head_dim), dtype=torch.float64, device="cuda")
    sum_do, sum_dv, sum_dk, abs_dk = z(), z(), z(), z()
    qdq = kdk = scale = 0.0
    for r0 in range(0, N, chunk):                           # chunked: no full-size fp64 temporaries at 1M tokens
        r1 = min(N, r0 + chunk)
        sum_do += inp["do"][0, r0:r1].double().view(r1 - r0, w.heads_kv, g, w.head_dim).sum((0, 2))
        dk = buf.dK[0, r0:r1].double()
        sum_dv += buf.dV[0, r0:r1].double().sum(0)
        sum_dk += dk.sum(0)
        abs_dk += dk.abs().sum(0)
        x = inp["q"][0, r0:r1].double() * buf.dQ[0, r0:r1].double()
        qdq += x.sum().item()
        scale += x.abs().sum().item()
        kdk += (inp["k"][0, r0:r1].double() * dk).sum().item()
    tol = TOL_GRAD * max(1.0, N ** 0.5 / 8)                 # N terms of per-element error add up like sqrt(N)
    assert (sum_dv - sum_do).abs().max().item() <= tol + 4e-3 * sum_do.abs().max().item()
    assert sum_dk.abs().max().item() <= tol + 4e-3 * abs_dk.max().item() / N ** 0.5
    assert abs(qdq - kdk) <= 1e-3 * scale


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_full_size_sampled(oracle, name):
    from paper_2512_20968_b200 import Buffers, plan_for

    w = W.CONFIGS[name]
    g = w.heads_q // w.heads_kv
    inp = W.make_inputs(w, "cuda")
    plan = plan_for(w, precision=1 if w.outlier else 0)
    buf = Buffers(plan, w, backward=True)
    rng = np.random.default_rng(100 + w.index)

    def run(do):
        plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
        plan.backward(inp["q"], inp["k"], inp["v"], buf.O, do, buf.lse, buf.bwd_ws, buf.dQ, buf.dK, buf.dV)
        torch.cuda.synchronize()

    run(inp["do"])

    # the oracle sees the last KV head and its group of query heads (GQA mapping h -> h / g stays valid on the slice)
    hk = w.heads_kv - 1
    q, do = _sub_bits(inp["q"], hk * g, (hk + 1) * g), _sub_bits(inp["do"], hk * g, (hk + 1) * g)
    k, v = _sub_bits(inp["k"], hk, hk + 1), _sub_bits(inp["v"], hk, hk + 1)
    pos = oracle.positions(w.n, w.L, w.seq_layout)

    # ---- sampled query rows of every Q partition: O, LSE, dQ
    parts = np.arange(w.n) if w.n <= 16 else np.unique(np.concatenate([np.arange(0, w.n, 5), [w.n - 1]]))
    rows = np.unique(np.concatenate([[p * w.L, p * w.L + w.L - 1, p * w.L + int(rng.integers(1, w.L - 1))] for p in parts]))
    hh = np.repeat(np.arange(g, dtype=np.int32), len(rows))
    rr = np.tile(rows, g)
    O_ref, lse_ref = oracle.fwd_rows(q, k, v, w.scale, w.causal, pos, rr, hh)
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, rr, hh)
    rows_t = torch.as_tensor(rows, device="cuda")
    O_g = buf.O[0, rows_t, hk * g:(hk + 1) * g].permute(1, 0, 2).reshape(-1, w.head_dim).cpu().numpy().astype(np.float64)
    dq_g = buf.dQ[0, rows_t, hk * g:(hk + 1) * g].permute(1, 0, 2).reshape(-1, w.head_dim).cpu().numpy().astype(np.float64)
    lse_g = buf.lse[0, hk * g:(hk + 1) * g][:, rows_t].reshape(-1).cpu().numpy().astype(np.float64)
    eO = np.abs(O_g - O_ref)
    assert np.isfinite(O_g).all() and np.isfinite(dq_g).all()
    assert eO.max() <= TOL_O_MAX and eO.mean() <= TOL_O_MEAN, (eO.max(), eO.mean())
    assert np.abs(lse_g - lse_ref).max() <= TOL_LSE
    assert np.abs(dq_g - dq_ref).max() <= TOL_GRAD, np.abs(dq_g - dq_ref).max()

    _invariants(w, inp, buf)

    # ---- dK, dV
    if w.causal:
        tail = np.where(pos >= w.seq_total - TAIL)[0]                  # rows holding the last TAIL token positions
        dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, True, pos, tail, np.zeros(len(tail), np.int32), qs_rows=tail)
        krows = tail
    else:
        live = np.unique(rng.integers(0, w.seq_total, 40))
        mask = torch.zeros(w.seq_total, dtype=torch.bool, device="cuda")
        mask[torch.as_tensor(live, device="cuda")] = True
        do_sparse = inp["do"] * mask[None, :, None, None]
        run(do_sparse)
        krows = np.unique(rng.integers(0, w.seq_total, 256))
        do_s = _sub_bits(do_sparse, hk * g, (hk + 1) * g)
        dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do_s, w.scale, False, pos, krows, np.zeros(len(krows), np.int32), qs_rows=live)
        assert torch.all(buf.dQ[0][~mask] == 0)                        # rows with dO = 0 have dQ = 0 exactly
    kr = torch.as_tensor(krows, device="cuda")
    dk_g = buf.dK[0, kr, hk].cpu().numpy().astype(np.float64)
    dv_g = buf.dV[0, kr, hk].cpu().numpy().astype(np.float64)
    assert np.abs(dk_g - dk_ref).max() <= TOL_GRAD, np.abs(dk_g - dk_ref).max()
    assert np.abs(dv_g - dv_ref).max() <= TOL_GRAD, np.abs(dv_g - dv_ref).max()
