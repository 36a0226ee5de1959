"""N > 1 path on the CPU (gloo, world_size 2).  The hot path does not shard (BASELINE.json: no sharding, no
collectives; replicas only), so the multi-rank logic is bench.py's bookkeeping: every rank
builds the same plan, the job time is the max over ranks, the job value is the sum of the ranks' work over that time,
and the oracle arm runs on rank 0 only.  The method's own sharding (paper_2512_20968_b200/distributed.py)
is driven here with stand-in compute: the collectives, groups and slot order of Alg.2 / Alg.3 on 2 and 4 gloo ranks."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2512_20968_b200 import binding as B
    from paper_2512_20968_b200 import plan_for
    from paper_2512_20968_b200 import workloads as W

    # every rank plans the same replica: identical assignment matrix, tile order and FLOP count
    w = W.scaled_down(W.C5, 256, heads_q=2)
    plan = plan_for(w)
    sig = torch.tensor([int(plan.am().astype("int64").sum()), int(plan.tiles(3).astype("int64").sum()),
                        plan.query(B.Q_FLOPS_FWD), plan.query(B.Q_FLOPS_BWD)], dtype=torch.int64)
    gathered = [torch.zeros_like(sig) for _ in range(world)]
    dist.all_gather(gathered, sig)
    assert all(torch.equal(g, sig) for g in gathered)

    # job time = slowest rank; job value = all ranks' work / that time
    ms = bench.max_over_ranks(100.0 * (rank + 1), dist, "cpu")
    assert ms == 100.0 * world
    flops = float(plan.query(B.Q_FLOPS_FWD) + plan.query(B.Q_FLOPS_BWD))
    val = bench.whole_job_tflops(flops, world, 2, ms)
    assert abs(val - world * flops * 2 / (ms / 1e3) / 1e12) < 1e-12 * val
    Path(out_dir, f"rank{rank}.json").write_text(json.dumps({"ms": ms, "value": val}))
    dist.barrier()
    dist.destroy_process_group()


def test_gloo_world2_bookkeeping(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    res = [json.loads((tmp_path / f"rank{r}.json").read_text()) for r in range(world)]
    assert res[0] == res[1]


def test_reference_arm_runs_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 prints the JSON line, rank 1 exits 0 without work."""
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29555")
        r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "C1", "--steps", "1",
                            "--warmup", "1", "--cpu-seconds", "0.5"], env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert outs[1] == ""


def _mesh_worker(rank: int, world: int, port: int, a: int, b: int, causal: bool, heads_q: int, heads_kv: int, out_dir: str):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.set_num_threads(2)
    from paper_2512_20968_b200 import plan_for
    from paper_2512_20968_b200 import workloads as W
    from tests.rank_standin import StandInKernels, StandInRank

    L, D = 128, 64
    w = W.Workload("mesh", 7, causal, a, b, 1, L * a * b, heads_q, heads_kv, D, seq_layout="striped" if causal else "contiguous")
    plan = plan_for(w)
    inp = W.make_inputs(w, "cpu")                                # same seed on every rank
    own = {k: v[:, rank * L:(rank + 1) * L].contiguous() for k, v in inp.items()}
    me = StandInRank(plan, StandInKernels(plan, w.seq_layout))
    O, lse = me.forward(own["q"], own["k"], own["v"])
    dQ, dK, dV = me.backward(own["do"])
    torch.save({"O": O, "lse": lse, "dQ": dQ, "dK": dK, "dV": dV}, Path(out_dir, f"rank{rank}.pt"))
    dist.barrier()
    dist.destroy_process_group()


def _check_mesh(tmp_path, a, b, causal, heads_q, heads_kv):
    from paper_2512_20968_b200 import workloads as W

    world, L, D = a * b, 128, 64
    mp.spawn(_mesh_worker, args=(world, _free_port(), a, b, causal, heads_q, heads_kv, str(tmp_path)), nprocs=world, join=True)
    res = [torch.load(tmp_path / f"rank{r}.pt") for r in range(world)]
    got = {k: torch.cat([r[k] for r in res], dim=2 if k == "lse" else 1).double() for k in res[0]}
    # full attention and its gradients from the definition (torch fp64 autograd), global token order via the position map
    w = W.Workload("mesh", 7, causal, a, b, 1, L * world, heads_q, heads_kv, D, seq_layout="striped" if causal else "contiguous")
    inp = {k: v.double() for k, v in W.make_inputs(w, "cpu").items()}
    q, k, v = (inp[x].clone().requires_grad_(True) for x in ("q", "k", "v"))
    p, s = torch.arange(w.seq_total) // L, torch.arange(w.seq_total) % L
    pos = s * world + p if causal else p * L + s
    grp = heads_q // heads_kv
    S = torch.einsum("bshd,bthd->bhst", q, k.repeat_interleave(grp, dim=2)) * w.scale
    if causal:
        S = S.masked_fill(pos[None, :] > pos[:, None], float("-inf"))
    O = torch.einsum("bhst,bthd->bshd", torch.softmax(S, -1), v.repeat_interleave(grp, dim=2))
    O.backward(inp["do"])
    ref = {"O": O.detach(), "lse": torch.logsumexp(S, -1).detach(), "dQ": q.grad, "dK": k.grad, "dV": v.grad}
    for name in ref:
        err = (got[name] - ref[name]).abs().max().item()
        assert err < 2e-4, f"{name}: max abs error {err:.3e} (fp32 buffers between the steps)"


def test_mesh_ranks_world2_q_group(tmp_path):
    """a = 2, b = 1: one Q group of two ranks (AG-Q, RS-O, RS-dQ carry data; the KV groups are singletons)."""
    _check_mesh(tmp_path, 2, 1, True, 2, 2)


def test_mesh_ranks_world2_kv_group(tmp_path):
    """a = 1, b = 2: one KV group of two ranks (AG-KV, RS-dKV); GQA 4 query heads on 2 KV heads."""
    _check_mesh(tmp_path, 1, 2, False, 4, 2)


def test_mesh_ranks_world4(tmp_path):
    """2 x 2 mesh, causal, striped: both group kinds, KV partition rotation (KV group of rank g = {g mod a + t*a})."""
    _check_mesh(tmp_path, 2, 2, True, 2, 1)


def test_mesh_groups_follow_the_assignment_matrix():
    """Q group of rank g = the ranks of its tile row, KV group = the ranks sharing its rotated KV footprint (PAPER.md L116,
    L157-161): both contain g, partition the ranks, and every (i, j) cell of the AM is owned by the one rank that sits in
    i's Q group and j's KV group.  Without KV rotation, or with a world size other than n, the mapping is refused."""
    import numpy as np
    import pytest

    from paper_2512_20968_b200 import plan_for
    from paper_2512_20968_b200 import workloads as W
    from paper_2512_20968_b200.distributed import mesh_groups

    for a, b in ((2, 2), (3, 3), (2, 4), (4, 2)):
        w = W.Workload("m", 7, True, a, b, 1, 128 * a * b, 2, 2, 64, seq_layout="striped")
        plan = plan_for(w)
        qg, kg = mesh_groups(plan, a * b)
        am = plan.am()
        assert sorted(set(map(tuple, qg))) == [tuple(range(r * a, (r + 1) * a)) for r in range(b)]
        assert sorted(set(map(tuple, kg))) == [tuple(c + t * a for t in range(b)) for c in range(a)]
        for i in range(a * b):
            for j in range(a * b):
                owners = [g for g in range(a * b) if i in qg[g] and j in kg[g]]
                assert owners == [int(am[i, j])]
        with pytest.raises(ValueError):
            mesh_groups(plan, a * b + 1)
    w = W.Workload("m", 7, False, 2, 2, 1, 512, 2, 2, 64, kvr=False)
    with pytest.raises(ValueError):
        mesh_groups(plan_for(w), 4)


def test_bench_reads_roofline_traffic_from_profiles():
    """roofline.traffic comes from an ncu capture under profiles/ (never from a constant in bench.py), with the commit and the
    kernel-source hash it was taken at; a workload without a capture gets null and a reason."""
    sys.path.insert(0, str(ROOT))
    import bench
    from paper_2512_20968_b200.build import kernel_source_hash

    traffic, src = bench.load_traffic("C5", "tile_bwd")
    assert traffic and traffic == src["dram_read_bytes"] + src["dram_write_bytes"]
    assert src["file"].startswith("profiles/") and (ROOT / src["file"]).exists()
    assert src["kernel_sha16_now"] == kernel_source_hash("tile_bwd") and len(src["kernel_sha16_now"]) == 16
    assert isinstance(src["matches_current_kernel"], bool) and src["commit"]
    none, why = bench.load_traffic("C3", "tile_bwd")
    assert none is None and "reason" in why
