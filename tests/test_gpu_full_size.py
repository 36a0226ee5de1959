"""GPU parity at BASELINE.json's FULL sizes (configs[1..4]), in the launch configuration bench.py times
(mesh_attn_forward + mesh_attn_backward through the C ABI), on outputs the fp64 oracle can compute one by one
(the method's backward is PAPER.md L236, Alg.3):

  1. O, LSE and dQ on sampled query rows of EVERY Q partition (first / last / one random local row of each of the n
     partitions): a row costs the oracle 4*N*D + 6*N*D flops per head, and the sample touches every simulated GPU and
     every (Q_u, KV_v) pair;
  2. causal configs: dK, dV of the keys at the last TAIL = 256 token positions, which only the last 256 queries see --
     exact with 256 oracle rows (under the striped layout they live in 256 / n .. 256 different partitions);
  3. EVERY config (causal ones included): the sparse-dO probe -- a second backward with dO non-zero on R = 40 query
     rows spread over the partitions (gradients are linear in dO, so ALL of dK, dV depends on R oracle rows): dK, dV
     compared element-wise on >= 256 sampled keys drawn from EVERY KV partition, from the first, a middle and the last
     128-key block of a partition, and dQ == 0 exactly on the rows whose dO is zero;
  4. properties that hold at any size: sum_t dV = sum_s dO, sum_t dK = 0, <Q,dQ> = <K,dK> (per KV head / globally).

Tolerances are BASELINE.json's.  configs[2] (outlier scores) runs with plan precision = 1.
The per-config maxima are printed (pytest -s / the captured output of the GPU run)."""
import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W
from tests.util import torch_bits

pytestmark = pytest.mark.gpu

TOL_O_MAX, TOL_O_MEAN, TOL_LSE, TOL_GRAD = 1e-2, 1e-3, 1e-3, 2e-2
TAIL = 256         # causal: keys at the last TAIL token positions
PROBE_ROWS = 40    # sparse-dO probe: query rows with non-zero dO
PROBE_KEYS = 256   # sparse-dO probe: at least this many sampled keys, every KV partition represented


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


def _probe_rows(w, rng):
    """Query rows of the sparse-dO probe: spread over the partitions, early and late local rows, and (causal) a few rows
    at the very last token positions so that keys of every position receive from at least one live query."""
    parts = rng.choice(w.n, size=min(w.n, PROBE_ROWS - 8), replace=False)
    rows = [int(p) * w.L + int(rng.integers(0, w.L)) for p in parts]
    while len(rows) < PROBE_ROWS - 8:
        rows.append(int(rng.integers(0, w.seq_total)))
    late = rng.choice(w.n, size=min(w.n, 8), replace=False)
    rows += [int(p) * w.L + w.L - 1 - int(rng.integers(0, 4)) for p in late]     # local rows L-4..L-1: the last positions
    return np.unique(np.asarray(rows, dtype=np.int64))


def _probe_keys(w, rng):
    """Sampled key rows: every KV partition, its first / a middle / its last 128-key block, plus random rows."""
    per = max(3, -(-PROBE_KEYS // w.n))
    nblk = w.L // 128
    keys = []
    for p in range(w.n):
        loc = [int(rng.integers(0, 128)), (nblk // 2) * 128 + int(rng.integers(0, 128)), (nblk - 1) * 128 + int(rng.integers(0, 128))]
        loc = loc[p % 3:] + loc[:p % 3]                    # which of the three comes first rotates with the partition
        loc += [int(x) for x in rng.integers(0, w.L, max(0, per - 3))]
        keys += [p * w.L + s for s in loc[:per]]
    keys = np.unique(np.asarray(keys, dtype=np.int64))
    while len(keys) < PROBE_KEYS:                          # duplicates collapsed: top up with random rows
        keys = np.unique(np.concatenate([keys, rng.integers(0, w.seq_total, PROBE_KEYS - len(keys))]))
    return keys


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
    err = {}

    # ---- 1. sampled query rows of EVERY Q partition: O, LSE, dQ
    rows = np.unique(np.concatenate([[p * w.L, p * w.L + w.L - 1, p * w.L + int(rng.integers(1, w.L - 1))] for p in range(w.n)]))
    hh = np.repeat(np.arange(g, dtype=np.int32), len(rows))
    rr = np.tile(rows, g)
    O_ref, lse_ref = oracle.fwd_rows(q, k, v, w.scale, w.causal, pos, rr, hh)
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, rr, hh)
    rows_t = torch.as_tensor(rows, device="cuda")
    O_g = buf.O[0, rows_t, hk * g:(hk + 1) * g].permute(1, 0, 2).reshape(-1, w.head_dim).cpu().numpy().astype(np.float64)
    dq_g = buf.dQ[0, rows_t, hk * g:(hk + 1) * g].permute(1, 0, 2).reshape(-1, w.head_dim).cpu().numpy().astype(np.float64)
    lse_g = buf.lse[0, hk * g:(hk + 1) * g][:, rows_t].reshape(-1).cpu().numpy().astype(np.float64)
    eO = np.abs(O_g - O_ref)
    err.update(O_max=eO.max(), O_mean=eO.mean(), lse=np.abs(lse_g - lse_ref).max(), dQ=np.abs(dq_g - dq_ref).max(), rows=len(rows))
    assert np.isfinite(O_g).all() and np.isfinite(dq_g).all()
    assert err["O_max"] <= TOL_O_MAX and err["O_mean"] <= TOL_O_MEAN, err
    assert err["lse"] <= TOL_LSE, err
    assert err["dQ"] <= TOL_GRAD, err

    # ---- 4. whole-tensor properties
    _invariants(w, inp, buf)

    def grads_at(krows):
        kr = torch.as_tensor(krows, device="cuda")
        return buf.dK[0, kr, hk].cpu().numpy().astype(np.float64), buf.dV[0, kr, hk].cpu().numpy().astype(np.float64)

    # ---- 2. causal: dK, dV of the keys at the last TAIL token positions (dense dO)
    if w.causal:
        tail = np.where(pos >= w.seq_total - TAIL)[0]                  # rows holding the last TAIL token positions
        dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, True, pos, tail, np.zeros(len(tail), np.int32), qs_rows=tail)
        dk_g, dv_g = grads_at(tail)
        err.update(dK_tail=np.abs(dk_g - dk_ref).max(), dV_tail=np.abs(dv_g - dv_ref).max())
        assert err["dK_tail"] <= TOL_GRAD and err["dV_tail"] <= TOL_GRAD, err

    # ---- 3. sparse-dO probe: dK, dV element-wise on keys of every KV partition; dQ == 0 on the dead rows
    live = _probe_rows(w, rng)
    mask = torch.zeros(w.seq_total, dtype=torch.bool, device="cuda")
    mask[torch.as_tensor(live, device="cuda")] = True
    do_sparse = inp["do"] * mask[None, :, None, None]
    run(do_sparse)
    krows = _probe_keys(w, rng)
    assert len(krows) >= PROBE_KEYS and len(np.unique(krows // w.L)) == w.n
    do_s = _sub_bits(do_sparse, hk * g, (hk + 1) * g)
    dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do_s, w.scale, w.causal, pos, krows, np.zeros(len(krows), np.int32), qs_rows=live)
    dk_g, dv_g = grads_at(krows)
    err.update(dK_probe=np.abs(dk_g - dk_ref).max(), dV_probe=np.abs(dv_g - dv_ref).max(), probe_keys=len(krows),
               probe_ref_max=max(np.abs(dk_ref).max(), np.abs(dv_ref).max()))
    print(f"\n{name} full size: " + ", ".join(f"{k_}={v_:.3g}" for k_, v_ in err.items()))
    assert err["probe_ref_max"] > 0.0                                  # the probe is not vacuous
    assert err["dK_probe"] <= TOL_GRAD and err["dV_probe"] <= TOL_GRAD, err
    for r0 in range(0, w.seq_total, 1 << 16):                          # rows with dO = 0 have dQ = 0 exactly
        r1 = min(w.seq_total, r0 + (1 << 16))
        assert torch.all(buf.dQ[0, r0:r1][~mask[r0:r1]] == 0)
    # the live rows' dQ against the oracle (the same rows, sparse dO)
    lr = np.tile(live, g)
    lh = np.repeat(np.arange(g, dtype=np.int32), len(live))
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do_s, w.scale, w.causal, pos, lr, lh)
    live_t = torch.as_tensor(live, device="cuda")
    dq_g = buf.dQ[0, live_t, hk * g:(hk + 1) * g].permute(1, 0, 2).reshape(-1, w.head_dim).cpu().numpy().astype(np.float64)
    assert np.abs(dq_g - dq_ref).max() <= TOL_GRAD, np.abs(dq_g - dq_ref).max()
