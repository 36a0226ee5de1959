"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path and the oracle tests and therefore holds none of
the method's arithmetic: only the configuration table (BASELINE.json ``configs``) and the
random bf16 tensors.  The paper's experiments are themselves synthetic attention calls
defined by shape only (BF16, batch 1, head_dim 128, 64 heads, 256K-1M tokens) and state no
value distribution; BASELINE.json's distributions stand in.

The bf16 *bits* are the ground truth: generate once (on whichever device), then copy the
bits to the other side; never regenerate independently on host and device.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import torch

SEED_BASE = 251220968          # arXiv id of the paper; seed of config k is SEED_BASE + k
OUTLIER_CHANNELS = (16, 48, 80, 112)
OUTLIER_SCALE = 8.0            # power of two: exact in bf16


@dataclass(frozen=True)
class Workload:
    name: str
    index: int                 # k in seed = SEED_BASE + k
    causal: bool
    a: int                     # tile height  = Q-group size
    b: int                     # tile width   = KV-group size
    batch: int
    seq_total: int
    heads_q: int
    heads_kv: int
    head_dim: int
    outlier: bool = False      # C3: 4 of 128 Q/K channels scaled x8
    kvr: bool = True           # KV partition rotation
    order: str = "row_major"   # "row_major" | "greedy"
    k_q: int = 1
    k_kv: int = 1
    seq_layout: str = "contiguous"   # causal configs use "striped"
    backward: bool = True

    @property
    def n(self) -> int:
        return self.a * self.b

    @property
    def L(self) -> int:
        return self.seq_total // self.n

    @property
    def scale(self) -> float:
        return self.head_dim ** -0.5

    def visible_pairs(self) -> int:
        N = self.seq_total
        return N * (N + 1) // 2 if self.causal else N * N

    def flops_fwd(self) -> float:
        """Algorithmic forward FLOPs: 4*D per visible (q,k) pair per query head."""
        return 4.0 * self.head_dim * self.heads_q * self.batch * self.visible_pairs()

    def flops_bwd(self) -> float:
        """Algorithmic backward FLOPs: 10*D per visible pair per query head (5 GEMMs)."""
        return 10.0 * self.head_dim * self.heads_q * self.batch * self.visible_pairs()


# BASELINE.json configs[0..4]
C1 = Workload("C1", 1, False, 2, 2, 1, 1024, 4, 4, 64, backward=False)
C2 = Workload("C2", 2, False, 3, 3, 1, 36864, 32, 32, 128)
C3 = Workload("C3", 3, True, 4, 4, 1, 131072, 32, 32, 128, outlier=True, order="greedy", k_q=2, k_kv=2,
              seq_layout="striped")
C4 = Workload("C4", 4, True, 8, 8, 1, 262144, 32, 8, 128, seq_layout="striped")
C5 = Workload("C5", 5, True, 16, 16, 1, 1048576, 32, 32, 128, order="greedy", k_q=2, k_kv=2,
              seq_layout="striped")
CONFIGS = {w.name: w for w in (C1, C2, C3, C4, C5)}


def scaled_down(w: Workload, L: int, heads_q: int | None = None, heads_kv: int | None = None) -> Workload:
    """Same structure (mesh, mask, GQA ratio, distribution, order) with a smaller partition length / head count."""
    hq = w.heads_q if heads_q is None else heads_q
    hkv = (hq * w.heads_kv // w.heads_q) if heads_kv is None else heads_kv
    return replace(w, name=f"{w.name}s", seq_total=L * w.n, heads_q=hq, heads_kv=max(1, hkv))


def _randn_bf16(shape, seed: int, device, outlier: bool, chunk_rows: int = 1 << 15) -> torch.Tensor:
    """iid N(0,1) in fp32 -> optional x8 on OUTLIER_CHANNELS -> round-to-nearest-even bf16. shape = [B, N, H, D]."""
    B, N, H, D = shape
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed)
    out = torch.empty(shape, dtype=torch.bfloat16, device=dev)
    flat = out.view(B * N, H, D)
    for r0 in range(0, B * N, chunk_rows):
        r1 = min(B * N, r0 + chunk_rows)
        x = torch.randn((r1 - r0, H, D), generator=gen, device=dev, dtype=torch.float32)
        if outlier:
            x[..., list(c for c in OUTLIER_CHANNELS if c < D)] *= OUTLIER_SCALE
        flat[r0:r1] = x.to(torch.bfloat16)
    return out


def make_inputs(w: Workload, device="cpu", which=("q", "k", "v", "do")) -> dict:
    """Seeded bf16 tensors, layout [B, N, H, D], rows partition-major (row = p*L + s)."""
    seed = SEED_BASE + w.index
    spec = {
        "q": ((w.batch, w.seq_total, w.heads_q, w.head_dim), 0, w.outlier),
        "k": ((w.batch, w.seq_total, w.heads_kv, w.head_dim), 1, w.outlier),
        "v": ((w.batch, w.seq_total, w.heads_kv, w.head_dim), 2, False),
        "do": ((w.batch, w.seq_total, w.heads_q, w.head_dim), 3, False),
    }
    return {name: _randn_bf16(spec[name][0], seed * 16 + spec[name][1], device, spec[name][2]) for name in which}
