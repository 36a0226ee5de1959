"""Test-side stand-in for the four per-rank kernels (plain torch fp64 on the CPU, written from the definition of
attention and its gradients): lets the gloo tests drive paper_2512_20968_b200.distributed.MeshAttnRank -- group
construction, slot order, routing of the partials, reduce-scatters -- on a box without a GPU.  Not a product path."""
import math

import torch

from paper_2512_20968_b200.distributed import MeshAttnRank


class StandInRank(MeshAttnRank):
    """MeshAttnRank with its compute calls replaced by the stand-in below: the product class takes no such argument."""

    def __init__(self, plan, standin, **kw):
        super().__init__(plan, **kw)
        self._kernels = standin


class StandInKernels:
    def __init__(self, plan, seq_layout: str):
        d = plan.desc
        self.plan, self.n, self.a, self.b = plan, d.n, d.a, d.b
        self.L, self.Hq, self.Hkv, self.D = d.seq_total // d.n, d.heads_q, d.heads_kv, d.head_dim
        self.causal, self.striped = bool(d.causal), seq_layout == "striped"
        self.scale = d.softmax_scale if d.softmax_scale > 0 else d.head_dim ** -0.5

    def _pos(self, parts):
        s = torch.arange(self.L)
        return torch.cat([(s * self.n + int(p)) if self.striped else (int(p) * self.L + s) for p in parts])

    def _scores(self, g, Q_loc, K_loc):
        iq, ikv = self.plan.footprint(g)
        q = Q_loc.double()                                             # [B, a*L, Hq, D]
        k = K_loc.double().repeat_interleave(self.Hq // self.Hkv, dim=2)
        S = torch.einsum("bshd,bthd->bhst", q, k) * self.scale
        if self.causal:
            vis = self._pos(ikv)[None, :] <= self._pos(iq)[:, None]
            S = S.masked_fill(~vis, float("-inf"))
        return S

    def rank_fwd(self, g, Q_loc, K_loc, V_loc, partial_O, partial_lse):
        S = self._scores(g, Q_loc, K_loc)                              # [B, Hq, a*L, b*L]
        lse = torch.logsumexp(S, dim=-1)                               # -inf where nothing is visible
        P = torch.exp(S - torch.where(torch.isinf(lse), torch.zeros_like(lse), lse)[..., None])
        v = V_loc.double().repeat_interleave(self.Hq // self.Hkv, dim=2)
        O = torch.einsum("bhst,bthd->bshd", P, v)
        B = Q_loc.shape[0]
        partial_O.copy_(O.view(B, self.a, self.L, self.Hq, self.D).transpose(0, 1))
        partial_lse.copy_(lse.view(B, self.Hq, self.a, self.L).permute(2, 0, 1, 3))

    def rank_merge(self, recv_O, recv_lse, O_own, lse_own):
        lse = torch.logsumexp(recv_lse.double(), dim=0)                # [B, Hq, L]
        w = torch.exp(recv_lse.double() - torch.where(torch.isinf(lse), torch.zeros_like(lse), lse)[None])
        O_own.copy_((w.permute(0, 1, 3, 2)[..., None] * recv_O.double()).sum(0))
        lse_own.copy_(lse)

    def rank_bwd_preprocess(self, O_own, dO_own, lse_own, ws_own):
        ws_own[0].copy_((O_own.double() * dO_own.double()).sum(-1).permute(0, 2, 1))
        ws_own[1].copy_(math.log2(self.scale) - lse_own.double() * math.log2(math.e))

    def rank_bwd(self, g, Q_loc, K_loc, V_loc, dO_loc, ws_loc, dQ_loc, dK_loc, dV_loc):
        grp = self.Hq // self.Hkv
        S = self._scores(g, Q_loc, K_loc)
        lse = (math.log2(self.scale) - ws_loc[1].double()) / math.log2(math.e)     # [B, Hq, a*L]
        P = torch.exp(S - lse[..., None])
        do = dO_loc.double()
        v = V_loc.double().repeat_interleave(grp, dim=2)
        k = K_loc.double().repeat_interleave(grp, dim=2)
        dP = torch.einsum("bshd,bthd->bhst", do, v)
        dS = P * (dP - ws_loc[0].double()[..., None])
        B, bL = K_loc.shape[0], K_loc.shape[1]
        dV = torch.einsum("bhst,bshd->bthd", P, do).view(B, bL, self.Hkv, grp, self.D).sum(3)
        dK = self.scale * torch.einsum("bhst,bshd->bthd", dS, Q_loc.double()).view(B, bL, self.Hkv, grp, self.D).sum(3)
        dQ_loc += (self.scale * torch.einsum("bhst,bthd->bshd", dS, k)).float()
        dK_loc += dK.float()
        dV_loc += dV.float()
