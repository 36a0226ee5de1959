"""Plumbing around the C-ABI calls: plan construction from a Workload and device buffers.
No arithmetic of the method lives here."""
from __future__ import annotations

import torch

from .binding import Plan, Q_BWD_WS_BYTES, Q_PARTIAL_LSE_BYTES, Q_PARTIAL_O_BYTES
from .workloads import Workload


def plan_for(w: Workload, **overrides) -> Plan:
    kw = dict(
        a=w.a, b=w.b, n=w.n, batch=w.batch, seq_total=w.seq_total, heads_q=w.heads_q, heads_kv=w.heads_kv, head_dim=w.head_dim,
        causal=int(w.causal), kvr=int(w.kvr), seq_layout=int(w.seq_layout == "striped"), order=int(w.order == "greedy"),
        k_q=w.k_q, k_kv=w.k_kv,
        precision=1 if w.outlier else 0,   # outlier scores (BASELINE.json configs[2]) need hi+lo P / dS operands for the gradient bar
    )
    kw.update(overrides)
    return Plan(**kw)


class Buffers:
    """Caller-owned device buffers for one workload (the library never allocates in hot calls)."""

    def __init__(self, plan: Plan, w: Workload, backward: bool = True, g_count: int | None = None, device="cuda"):
        B, N, Hq, Hkv, D = w.batch, w.seq_total, w.heads_q, w.heads_kv, w.head_dim
        g_count = w.a if g_count is None else g_count
        f32 = dict(dtype=torch.float32, device=device)
        self.partial_O = torch.empty(plan.query(Q_PARTIAL_O_BYTES) * g_count // 4, **f32)
        self.partial_lse = torch.empty(plan.query(Q_PARTIAL_LSE_BYTES) * g_count // 4, **f32)
        out = dict(dtype=torch.bfloat16 if plan.desc.out_dtype == 1 else torch.float32, device=device)   # plan desc field out_dtype
        self.O = torch.empty((B, N, Hq, D), **out)
        self.lse = torch.empty((B, Hq, N), **f32)
        if backward:
            # [0] = delta, [1] = log2(scale) - lse*log2(e); out_dtype 1: the fp32 accumulators of dQ, dK, dV follow (Q_BWD_WS_BYTES)
            self.bwd_ws = torch.empty(plan.query(Q_BWD_WS_BYTES) // 4, **f32)
            self.delta = self.bwd_ws[:B * Hq * N].view(B, Hq, N)
            self.dQ = torch.empty((B, N, Hq, D), **out)
            self.dK = torch.empty((B, N, Hkv, D), **out)
            self.dV = torch.empty((B, N, Hkv, D), **out)
