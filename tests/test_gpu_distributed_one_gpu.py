"""The multi-GPU code of SURVEY.md 8(f).4 EXECUTED on the one B200 a box has (VERDICT r1 "Execute the f.4 code that has never run"):

  (a) ``distributed.MeshAttnRank`` end to end as a ONE-rank NCCL job (a = b = n = 1), both forms: ``peer_memory=False`` (NCCL
      sub-communicators, all-gathers, all-to-all, reduce-scatter) and ``peer_memory=True`` (``symm_mem.empty`` / ``rendezvous`` /
      ``barrier``, ``mesh_attn_rank_merge_peers`` and ``mesh_attn_rank_sum_peers`` on the symmetric-memory handles' pointers),
      forward and backward against the fp64 oracle (Alg.2, Alg.3; groups L178-182);
  (b) the peer-memory reducers on pointers that belong to ANOTHER PROCESS: a second process on the same GPU writes member 1's
      partials / gradient slots, exports them through CUDA IPC, and this process reads them in place (a = 2): bit-identical to
      the same reducer on a local copy, and equal to the oracle's merge.

Each case runs in a subprocess of its own (a process group / a CUDA IPC mapping must not leak into the other GPU tests).  No
kernel of one process waits on a kernel of the other (B200_PROFILING.md): the producer process has finished and synchronised
before the consumer launches anything."""
import os
import socket
import subprocess
import sys
import textwrap
from pathlib import Path

import pytest

pytestmark = pytest.mark.gpu
ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _run(code: str, timeout=600):
    import tempfile

    with tempfile.TemporaryDirectory() as tmp:             # a real file: multiprocessing's spawn re-imports the main module
        script = Path(tmp) / "one_gpu_case.py"
        script.write_text(textwrap.dedent(code))
        return _run_script(script, timeout)


def _run_script(script: Path, timeout):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()), RANK="0", WORLD_SIZE="1", LOCAL_RANK="0",
               PYTHONPATH=str(ROOT) + os.pathsep + os.environ.get("PYTHONPATH", ""))
    r = subprocess.run([sys.executable, str(script)], capture_output=True, text=True, env=env, timeout=timeout, cwd=str(ROOT))
    assert r.returncode == 0, r.stdout[-3000:] + "\n" + r.stderr[-6000:]
    return r.stdout


ONE_RANK = """
    import numpy as np, torch, torch.distributed as dist
    from dataclasses import replace
    from oracle import attn_oracle as oracle
    from paper_2512_20968_b200 import plan_for, launch_count
    from paper_2512_20968_b200 import workloads as W
    from paper_2512_20968_b200.distributed import MeshAttnRank

    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    peer = {peer}
    causal = {causal}
    w = W.Workload("one", 9, causal, 1, 1, 1, 512, 4, 2, 128, seq_layout="striped" if causal else "contiguous")
    plan = plan_for(w)
    inp = W.make_inputs(w, "cuda")
    me = MeshAttnRank(plan, peer_memory=peer)
    n0 = launch_count()
    for it in range(2):                                    # twice: the symmetric buffers and their barriers are reused
        O, lse = me.forward(inp["q"], inp["k"], inp["v"])
        dQ, dK, dV = me.backward(inp["do"])
    torch.cuda.synchronize()
    assert launch_count() - n0 >= 2 * (4 + (3 if peer else 0)), launch_count() - n0
    plan.health()
    bits = lambda t: t[0].cpu().contiguous().view(torch.int16).numpy().view(np.uint16)
    q, k, v, do = (bits(inp[x]) for x in ("q", "k", "v", "do"))
    pos = oracle.positions(1, w.L, w.seq_layout)
    rows = np.arange(w.seq_total, dtype=np.int64)
    rr, hh = np.repeat(rows, w.heads_q), np.tile(np.arange(w.heads_q, dtype=np.int32), len(rows))
    O_ref, lse_ref = oracle.fwd_rows(q, k, v, w.scale, w.causal, pos, rr, hh)
    dq_ref, _, _ = oracle.bwd_dq_rows(q, k, v, do, w.scale, w.causal, pos, rr, hh)
    kr, kh = np.repeat(rows, w.heads_kv), np.tile(np.arange(w.heads_kv, dtype=np.int32), len(rows))
    dk_ref, dv_ref = oracle.bwd_dkv_keys(q, k, v, do, w.scale, w.causal, pos, kr, kh)
    e_o = np.abs(O[0].cpu().numpy()[rr, hh] - O_ref)
    e_l = np.abs(lse[0].cpu().numpy()[hh, rr] - lse_ref).max()
    e_q = np.abs(dQ[0].cpu().numpy()[rr, hh] - dq_ref).max()
    e_k = np.abs(dK[0].cpu().numpy()[kr, kh] - dk_ref).max()
    e_v = np.abs(dV[0].cpu().numpy()[kr, kh] - dv_ref).max()
    print(f"one-rank job peer_memory={{peer}} causal={{causal}}: O {{e_o.max():.2e}} lse {{e_l:.2e}} dQ {{e_q:.2e}} dK {{e_k:.2e}} dV {{e_v:.2e}}")
    assert e_o.max() <= 1e-2 and e_o.mean() <= 1e-3 and e_l <= 1e-3 and max(e_q, e_k, e_v) <= 2e-2
    dist.destroy_process_group()
"""


@pytest.mark.parametrize("peer", [False, True])
@pytest.mark.parametrize("causal", [False, True])
def test_mesh_attn_rank_as_a_one_rank_nccl_job(peer, causal):
    print(_run(ONE_RANK.format(peer=peer, causal=causal)))


IPC = """
    import numpy as np, torch, torch.multiprocessing as mp

    def member_one(q, ready, done):
        # the OTHER process: member 1 of a Q group of two writes its partial (O, lse) for the consumer's partition and a
        # gradient slot, then hands the device buffers over by CUDA IPC (torch's reductions) and waits
        import torch
        torch.cuda.set_device(0)
        g = torch.Generator(device="cuda"); g.manual_seed(4242)
        B, L, Hq, D = 1, 256, 4, 128
        pO = torch.randn((B, L, Hq, D), generator=g, device="cuda")
        pl = torch.randn((B, Hq, L), generator=g, device="cuda") * 3
        pl[0, 1, 5] = float("-inf")                        # a row this member saw no key of (DESIGN.md reading R5)
        pO[0, 5, 1] = 0
        grad = torch.randn((L * Hq * D,), generator=g, device="cuda")
        torch.cuda.synchronize()                           # finished before the consumer launches anything
        q.put((pO, pl, grad))
        ready.set()
        done.wait(300)

    if __name__ == "__main__":
        mp.set_start_method("spawn", force=True)
        q, ready, done = mp.Queue(), mp.Event(), mp.Event()
        p = mp.Process(target=member_one, args=(q, ready, done))
        p.start()
        try:
            from oracle import attn_oracle as oracle
            from paper_2512_20968_b200 import plan_for
            from paper_2512_20968_b200 import workloads as W

            torch.cuda.set_device(0)
            assert ready.wait(300)
            fO, fl, fgrad = q.get(timeout=60)              # tensors backed by the OTHER process's allocations
            B, L, Hq, D = 1, 256, 4, 128
            w = W.Workload("ipc", 10, False, 2, 1, B, 2 * L, Hq, Hq, D)
            plan = plan_for(w)
            g = torch.Generator(device="cuda"); g.manual_seed(77)
            mO = torch.randn((B, L, Hq, D), generator=g, device="cuda")         # member 0 = this process
            ml = torch.randn((B, Hq, L), generator=g, device="cuda") * 3
            mgrad = torch.randn((L * Hq * D,), generator=g, device="cuda")
            O_p, lse_p = torch.empty_like(mO), torch.empty_like(ml)
            plan.rank_merge_peers([mO, fO], [ml, fl], O_p, lse_p)               # member 1's partial read IN PLACE, foreign memory
            recv_O, recv_l = torch.stack([mO, fO.clone()]).contiguous(), torch.stack([ml, fl.clone()]).contiguous()
            O_l, lse_l = torch.empty_like(mO), torch.empty_like(ml)
            plan.rank_merge(recv_O, recv_l, O_l, lse_l)                         # the same reducer on a local copy
            s_p, s_l = torch.empty_like(mgrad), torch.empty_like(mgrad)
            plan.rank_sum_peers([mgrad, fgrad], s_p)
            plan.rank_sum_peers([mgrad, fgrad.clone()], s_l)
            torch.cuda.synchronize()
            assert torch.equal(O_p, O_l) and torch.equal(lse_p, lse_l), "merge over foreign pointers differs from the local merge"
            assert torch.equal(s_p, s_l) and torch.equal(s_p, mgrad + fgrad)
            # against the oracle's merge, row by row
            Oc, lc = recv_O.double().cpu().numpy(), recv_l.double().cpu().numpy()
            err = 0.0
            for (row, h) in [(0, 0), (5, 1), (17, 2), (255, 3), (128, 0)]:
                O_ref, l_ref = oracle.merge(Oc[:, 0, row, h, :], lc[:, 0, h, row])
                err = max(err, float(np.abs(O_p[0, row, h].double().cpu().numpy() - O_ref).max()), abs(float(lse_p[0, h, row]) - l_ref))
            print(f"CUDA IPC peers: merge and sum over another process's memory bit-identical to the local forms; max err vs oracle {err:.2e}")
            assert err <= 1e-5
        finally:
            done.set()
            p.join(60)
"""


def test_peer_reducers_on_another_process_memory_cuda_ipc():
    print(_run(IPC))
