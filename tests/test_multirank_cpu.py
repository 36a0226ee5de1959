"""N > 1 path on the CPU (gloo, world_size 2).  The hot path does not shard (BASELINE.json: no sharding, no
collectives; replicas only), so the multi-rank logic is bench.py's bookkeeping: every rank
builds the same plan, the job time is the max over ranks, the job value is the sum of the ranks' work over that time,
and the oracle arm runs on rank 0 only."""
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
