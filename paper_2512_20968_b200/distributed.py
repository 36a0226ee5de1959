"""Mesh-Attention across real GPUs: rank g of an n-rank job is GPU g of the paper's mesh.

Alg.2 and Alg.3 (L246-255) with the collectives issued through ``torch.distributed`` on the
sub-groups the assignment matrix defines, and every compute step in the library's kernels through the per-rank
C-ABI calls (``mesh_attn_rank_fwd / rank_merge / rank_bwd_preprocess / rank_bwd``, include/mesh_attn.h):

    forward   AG-Q  over the Q group  (a ranks)  ->  Q_loc  [B, a*L, Hq, D]
              AG-KV over the KV group (b ranks)  ->  K_loc, V_loc [B, b*L, Hkv, D]
              rank_fwd: one partial (O, lse) per Q partition of the footprint
              RS-O  over the Q group: all-to-all of the partials, then rank_merge = the online-softmax reducer
    backward  rank_bwd_preprocess on the own rows (delta, exponent offset)
              AG of dO and of (delta, offset) over the Q group  (Alg.3 l.1 lists Q, O, dO: the two [Hq, L] vectors
              replace the all-gather of O; Q_loc, K_loc, V_loc are kept from the forward)
              rank_bwd: this GPU's contribution to dQ of its Q partitions and dK, dV of its KV partitions
              RS-dQ (sum over the Q group), RS-dKV (sum over the KV group)

Two forms of the exchanges that FOLLOW a compute step (RS-O, RS-dQ, RS-dKV):
  * ``peer_memory=False``: NCCL collectives (all-to-all + rank_merge; reduce_scatter) -- the baseline;
  * ``peer_memory=True`` : the partial buffers live in symmetric memory (``torch.distributed._symmetric_memory``) and the
    reducer reads every member's partial where it was written, over NVLink (``mesh_attn_rank_merge_peers``,
    ``mesh_attn_rank_sum_peers``): the loads of the reducer ARE the transfer, there is no receive buffer and no
    separate collective.  Each partial is read exactly once, so peer reads cost no extra link traffic.  The all-gathers
    that PRECEDE a compute step stay NCCL copies into local HBM on purpose: every Q / K / V tile is re-read by dozens of
    work items, and peer memory is not cached in the reader's L2.
Neither form has run on more than one GPU (this build's boxes have one).  What has run: the per-rank kernels, the
peer-memory reducers included, on one B200 with the n ranks played one after the other (tests/test_gpu_rank_calls.py); this
class end to end, both forms, as a ONE-rank NCCL job on one B200 (a = b = 1: sub-communicators, all-gathers, all-to-all,
reduce-scatter, ``symm_mem.empty`` / ``rendezvous`` / ``barrier`` and the peer reducers through the symmetric-memory handles)
and the peer reducers on pointers that really belong to ANOTHER process (CUDA IPC between two processes on the one GPU)
(tests/test_gpu_distributed_one_gpu.py); the group construction / slot order / routing by world-size 2 and 4 gloo processes
with stand-in compute (tests/test_multirank_cpu.py).  Needs kvr = 1 (with KV partition rotation the ranks
that share a KV footprint are exactly the owners of its partitions, L157-161), usp_lanes = 1, tensor_layout 0.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def mesh_groups(plan, world_size: int):
    """Q group and KV group of every rank, as sorted global rank lists, from the plan's footprints (L116-133, L159)."""
    n = plan.desc.n
    if world_size != n:
        raise ValueError(f"world size {world_size} != n = a*b = {n}: rank g is GPU g of the mesh")
    if not plan.desc.kvr:
        raise ValueError("the multi-GPU path needs kvr = 1: without KV partition rotation the GPUs sharing a KV footprint do not own it")
    q_groups, kv_groups = [], []
    for g in range(n):
        iq, ikv = plan.footprint(g)
        q_groups.append([int(x) for x in iq])      # slot k of a query-shaped local tensor <- rank iq[k]
        kv_groups.append([int(x) for x in ikv])    # slot t of a key-shaped local tensor   <- rank ikv[t]
        if g not in q_groups[-1] or g not in kv_groups[-1]:
            raise ValueError(f"rank {g} is not in its own footprint")
    return q_groups, kv_groups


def _gather_slots(own: torch.Tensor, ranks, group) -> torch.Tensor:
    """all-gather of [B, L, H, D] over `group` -> [B, len(ranks)*L, H, D], slot k from ranks[k] (ranks sorted = group order)."""
    m = len(ranks)
    stage = torch.empty((m,) + tuple(own.shape), dtype=own.dtype, device=own.device)
    dist.all_gather(list(stage.unbind(0)), own.contiguous(), group=group)
    B, L = own.shape[0], own.shape[1]
    if B == 1:
        return stage.view(1, m * L, *own.shape[2:])
    return stage.transpose(0, 1).reshape(B, m * L, *own.shape[2:])


def _reduce_scatter_slots(loc: torch.Tensor, ranks, own_index: int, group) -> torch.Tensor:
    """sum over the group of [B, m*L, H, D], member k keeps slot k -> [B, L, H, D]"""
    m = len(ranks)
    B, mL = loc.shape[0], loc.shape[1]
    L = mL // m
    chunks = [loc[:, k * L:(k + 1) * L].contiguous() for k in range(m)]
    out = torch.empty_like(chunks[own_index])
    if dist.get_backend(group) == "nccl":
        dist.reduce_scatter(out, chunks, op=dist.ReduceOp.SUM, group=group)
    else:   # gloo has no reduce_scatter: one reduce per destination
        for k, c in enumerate(chunks):
            dist.reduce(c, dst=ranks[k], op=dist.ReduceOp.SUM, group=group)
        out.copy_(chunks[own_index])
    return out


def _exchange_slots(send: torch.Tensor, ranks, own_index: int, group) -> torch.Tensor:
    """all-to-all of [m, ...]: slot k goes to member k; returns [m, ...] with slot k received from member k"""
    recv = torch.empty_like(send)
    if dist.get_backend(group) == "nccl":
        dist.all_to_all_single(recv, send.contiguous(), group=group)
    else:   # gloo has no all-to-all: one scatter per source
        for k, src in enumerate(ranks):
            dist.scatter(recv[k], list(send.unbind(0)) if k == own_index else None, src=src, group=group)
    return recv


class MeshAttnRank:
    """One rank of the job.  Every compute step runs in the library's kernels through the plan's ``rank_*`` calls; there is
    no other path (the CPU tests of the routing subclass this in tests/rank_standin.py and replace ``_kernels`` there)."""

    def __init__(self, plan, rank: int | None = None, world_size: int | None = None, peer_memory: bool = False):
        self.plan = plan
        self.peer_memory = peer_memory
        self.g = dist.get_rank() if rank is None else rank
        world = dist.get_world_size() if world_size is None else world_size
        d = plan.desc
        if max(d.usp_lanes, 1) != 1 or d.tensor_layout != 0 or d.partial_mode != 0:
            raise ValueError("MeshAttnRank needs usp_lanes = 1, tensor_layout 0, partial_mode 0")
        self._kernels = plan
        self.a, self.b, self.n = d.a, d.b, d.n
        self.B, self.L, self.Hq, self.Hkv, self.D = d.batch, d.seq_total // d.n, d.heads_q, d.heads_kv, d.head_dim
        q_groups, kv_groups = mesh_groups(plan, world)
        self.q_ranks, self.kv_ranks = q_groups[self.g], kv_groups[self.g]
        self.q_index, self.kv_index = self.q_ranks.index(self.g), self.kv_ranks.index(self.g)
        # dist.new_group is collective over the whole job: every rank creates every group, in the same order
        self.q_group = self.kv_group = None
        for ranks in sorted({tuple(x) for x in q_groups}):
            grp = dist.new_group(list(ranks))
            if list(ranks) == self.q_ranks:
                self.q_group = grp
        for ranks in sorted({tuple(x) for x in kv_groups}):
            grp = dist.new_group(list(ranks))
            if list(ranks) == self.kv_ranks:
                self.kv_group = grp
        self._saved = None
        self._symm = None

    def _symmetric(self, dev):
        """symmetric-memory buffers of the peer-memory form, created and exchanged once (collective over each group)"""
        if self._symm is None:
            import torch.distributed._symmetric_memory as symm_mem

            a, b, B, L, Hq, Hkv, D = self.a, self.b, self.B, self.L, self.Hq, self.Hkv, self.D
            f32 = dict(dtype=torch.float32, device=dev)
            bufs = {"pO": ((a, B, L, Hq, D), self.q_group), "plse": ((a, B, Hq, L), self.q_group), "dQ": ((B, a * L, Hq, D), self.q_group),
                    "dK": ((B, b * L, Hkv, D), self.kv_group), "dV": ((B, b * L, Hkv, D), self.kv_group)}
            self._symm = {}
            for name, (shape, grp) in bufs.items():
                t = symm_mem.empty(*shape, **f32)
                self._symm[name] = (t, symm_mem.rendezvous(t, grp))
        return self._symm

    @staticmethod
    def _slot_ptrs(handle, members: int, slot: int, slot_elems: int):
        return [int(handle.buffer_ptrs[k]) + slot * slot_elems * 4 for k in range(members)]

    # Alg.2
    def forward(self, Q_own: torch.Tensor, K_own: torch.Tensor, V_own: torch.Tensor):
        """Q_own bf16 [B, L, Hq, D], K_own, V_own bf16 [B, L, Hkv, D] (this rank's partition) -> O_own fp32 [B, L, Hq, D], lse_own fp32 [B, Hq, L]"""
        a, B, L, Hq, D = self.a, self.B, self.L, self.Hq, self.D
        dev = Q_own.device
        Q_loc = _gather_slots(Q_own, self.q_ranks, self.q_group)          # l.1 AG-Q
        K_loc = _gather_slots(K_own, self.kv_ranks, self.kv_group)        # l.2 AG-KV
        V_loc = _gather_slots(V_own, self.kv_ranks, self.kv_group)
        O_own = torch.empty((B, L, Hq, D), dtype=torch.float32, device=dev)
        lse_own = torch.empty((B, Hq, L), dtype=torch.float32, device=dev)
        if self.peer_memory:
            (partial_O, hO), (partial_lse, hl) = self._symmetric(dev)["pO"], self._symmetric(dev)["plse"]
            hO.barrier()                                                                # the members have merged the previous step's partials
            self._kernels.rank_fwd(self.g, Q_loc, K_loc, V_loc, partial_O, partial_lse)  # l.3-5
            hO.barrier()                                                                # every member's partials are written
            self._kernels.rank_merge_peers(self._slot_ptrs(hO, a, self.q_index, B * L * Hq * D),     # l.6 RS-O fused into the reducer
                                          self._slot_ptrs(hl, a, self.q_index, B * Hq * L), O_own, lse_own)
        else:
            partial_O = torch.empty((a, B, L, Hq, D), dtype=torch.float32, device=dev)
            partial_lse = torch.empty((a, B, Hq, L), dtype=torch.float32, device=dev)
            self._kernels.rank_fwd(self.g, Q_loc, K_loc, V_loc, partial_O, partial_lse)      # l.3-5
            recv_O = _exchange_slots(partial_O, self.q_ranks, self.q_index, self.q_group)   # l.6 RS-O: slot k -> member k
            recv_lse = _exchange_slots(partial_lse, self.q_ranks, self.q_index, self.q_group)
            self._kernels.rank_merge(recv_O, recv_lse, O_own, lse_own)                       # ... with the online-softmax reducer
        self._saved = (Q_loc, K_loc, V_loc, O_own, lse_own)
        return O_own, lse_own

    # Alg.3
    def backward(self, dO_own: torch.Tensor):
        """dO_own bf16 [B, L, Hq, D] -> dQ_own fp32 [B, L, Hq, D], dK_own, dV_own fp32 [B, L, Hkv, D]"""
        if self._saved is None:
            raise RuntimeError("backward before forward")
        Q_loc, K_loc, V_loc, O_own, lse_own = self._saved
        a, b, B, L, Hq, Hkv, D = self.a, self.b, self.B, self.L, self.Hq, self.Hkv, self.D
        dev = dO_own.device
        ws_own = torch.empty((2, B, Hq, L), dtype=torch.float32, device=dev)
        self._kernels.rank_bwd_preprocess(O_own, dO_own.contiguous(), lse_own, ws_own)
        dO_loc = _gather_slots(dO_own, self.q_ranks, self.q_group)                       # l.1 (with Q_loc kept from the forward)
        ws_all = torch.empty((a, 2, B, Hq, L), dtype=torch.float32, device=dev)
        dist.all_gather(list(ws_all.unbind(0)), ws_own, group=self.q_group)
        ws_loc = ws_all.permute(1, 2, 3, 0, 4).reshape(2, B, Hq, a * L).contiguous()    # member k at rows k*L..
        if self.peer_memory:
            if B != 1:
                raise ValueError("peer_memory=True takes batch 1 (a rank's slot of a local gradient must be contiguous)")
            sm = self._symmetric(dev)
            (dQ_loc, hQ), (dK_loc, hK), (dV_loc, hV) = sm["dQ"], sm["dK"], sm["dV"]
            hQ.barrier(); hK.barrier()                                                  # the previous step's sums have been read
            for t in (dQ_loc, dK_loc, dV_loc):
                t.zero_()
            self._kernels.rank_bwd(self.g, Q_loc, K_loc, V_loc, dO_loc, ws_loc, dQ_loc, dK_loc, dV_loc)   # l.3-5
            hQ.barrier(); hK.barrier()
            dQ_own = torch.empty((B, L, Hq, D), dtype=torch.float32, device=dev)
            dK_own = torch.empty((B, L, Hkv, D), dtype=torch.float32, device=dev)
            dV_own = torch.empty((B, L, Hkv, D), dtype=torch.float32, device=dev)
            self._kernels.rank_sum_peers(self._slot_ptrs(hQ, a, self.q_index, L * Hq * D), dQ_own)        # l.6 RS-dQ as peer reads
            self._kernels.rank_sum_peers(self._slot_ptrs(hK, b, self.kv_index, L * Hkv * D), dK_own)      # l.7 RS-dKV
            self._kernels.rank_sum_peers(self._slot_ptrs(hV, b, self.kv_index, L * Hkv * D), dV_own)
            return dQ_own, dK_own, dV_own
        dQ_loc = torch.zeros((B, a * L, Hq, D), dtype=torch.float32, device=dev)
        dK_loc = torch.zeros((B, b * L, Hkv, D), dtype=torch.float32, device=dev)
        dV_loc = torch.zeros((B, b * L, Hkv, D), dtype=torch.float32, device=dev)
        self._kernels.rank_bwd(self.g, Q_loc, K_loc, V_loc, dO_loc, ws_loc, dQ_loc, dK_loc, dV_loc)   # l.3-5
        dQ_own = _reduce_scatter_slots(dQ_loc, self.q_ranks, self.q_index, self.q_group)             # l.6 RS-dQ
        dK_own = _reduce_scatter_slots(dK_loc, self.kv_ranks, self.kv_index, self.kv_group)          # l.7 RS-dKV
        dV_own = _reduce_scatter_slots(dV_loc, self.kv_ranks, self.kv_index, self.kv_group)
        return dQ_own, dK_own, dV_own
