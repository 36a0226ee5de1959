"""GPU parity on RANDOM plan geometries: seeded draws over mesh shape (a x b, also a != b and a or b = 1), partition length
(1..5 key blocks, so ragged against the 256-row forward items and the backward's pairing), heads / GQA group, head_dim,
mask and sequence layout, KV rotation, tile order with k_Q x k_KV chunks, batch and Mesh-USP lanes -- the combinations the
named BASELINE.json shapes do not reach.  Every draw runs mesh_attn_forward + mesh_attn_backward through the C ABI and is
compared with the fp64 oracle (forward: sampled rows of every partition incl. its first and last row, all heads; backward:
sampled query rows and keys, plus the three gradient invariants), tolerances of BASELINE.json.  The draw list is fixed by
the seeds below; `geometry(seed)` is also exercised on the CPU (tests/test_planner.py) so that an invalid draw shows there."""
from dataclasses import replace

import numpy as np
import pytest
import torch

from paper_2512_20968_b200 import workloads as W

SEEDS = list(range(20))


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
    return w, dict(usp_lanes=lanes)


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
