#!/usr/bin/env python
"""bench.py -- one "step" = one pass of the whole hot path (plan -> tile forward ->
merge, bwd preprocess -> tile backward with in-place reductions) over one synthetic workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference]

Prints ONE JSON line (rank 0).  `value` = algorithmic forward+backward attention TFLOP/s of the whole
job (all N GPUs: replicas of the same workload), inputs resident in HBM;
`e2e` = the same metric through mesh_attn_step_host (host buffers, H2D/D2H inside the timed region);
`roofline` = the dominant kernel (tile backward) against the measured dense-bf16 peak, timed per
launch with CUDA events inside the timed region (mesh_attn_profile_*); `cpu_baseline` = the fp64 oracle
on the host cores over a bounded sample.  `--impl reference` times the oracle only (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "attention_fwd_bwd_tflops"
UNIT = "TFLOP/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_traffic(workload: str, kernel: str):
    """roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of `kernel` on `workload`, read from the
    newest ncu capture under profiles/ (`*_traffic_<workload>_<kernel>.csv`, written by `ncu --csv --metrics dram__bytes_read.sum,
    dram__bytes_write.sum,...`; its sidecar `.md` names the command, the commit and the hash of the kernel sources it was taken
    at).  Nothing is embedded in this file: no capture -> (None, reason)."""
    import csv
    import re

    from paper_2512_20968_b200.build import kernel_source_hash

    files = sorted((ROOT / "profiles").glob(f"*_traffic_{workload.lower()}_{kernel}.csv"),
                   key=lambda f: [int(x) for x in re.findall(r"\d+", f.name)[:2]])
    if not files:
        return None, {"reason": f"no profiles/*_traffic_{workload.lower()}_{kernel}.csv capture for this workload and kernel"}
    f = files[-1]
    import io

    vals = {}
    with open(f, newline="") as fh:
        body = "".join(line for line in fh if line.startswith('"'))       # ncu prefixes the csv with ==PROF== / ==WARNING== lines
    if True:
        for row in csv.DictReader(io.StringIO(body)):
            try:
                vals[row["Metric Name"]] = float(row["Metric Value"].replace(",", ""))
            except (KeyError, ValueError, TypeError):
                continue
    if "dram__bytes_read.sum" not in vals or "dram__bytes_write.sum" not in vals:
        return None, {"reason": f"{f.name} holds no dram__bytes_read.sum / dram__bytes_write.sum"}
    src = {"file": f"profiles/{f.name}", "dram_read_bytes": vals["dram__bytes_read.sum"], "dram_write_bytes": vals["dram__bytes_write.sum"]}
    if "lts__t_sector_hit_rate.pct" in vals:
        src["l2_hit_pct"] = vals["lts__t_sector_hit_rate.pct"]
    side = f.with_suffix(".md")
    meta = side.read_text() if side.exists() else ""
    for key in ("commit", "kernel_sha16"):
        m = re.search(rf"^{key}:\s*(\S+)", meta, flags=re.M)
        src[key] = m.group(1) if m else "unrecorded (captured before the sidecar files existed)"
    src["kernel_sha16_now"] = kernel_source_hash(kernel)
    src["matches_current_kernel"] = src["kernel_sha16"] == src["kernel_sha16_now"]
    return vals["dram__bytes_read.sum"] + vals["dram__bytes_write.sum"], src


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5", help="C1..C5 (BASELINE.json configs[0..4]); default: the 1M-token causal config")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target duration of the oracle sample")
    ap.add_argument("--usp-lanes", type=int, default=1, help="Mesh-USP lanes U (PAPER.md L372-389): the partial workspace shrinks by U")
    ap.add_argument("--goo-executor", type=int, default=-1, metavar="R",
                    help="separate mode (not the driver's bench line): time the GOO executor (mesh_attn_forward_goo) on --workload with every "
                         "communication stand-in copied R times, overlapped vs serialised, against the fused forward")
    ap.add_argument("--fwd-pairing", type=int, default=0, choices=[0, 1],
                    help="plan desc field fwd_pairing (A/B runs): 0 auto (tile_fwd as CTA pairs with cta_group::2 MMAs where the plan allows), 1 single CTAs")
    ap.add_argument("--bwd-pairing", type=int, default=0, choices=[0, 1, 2],
                    help="plan desc field bwd_pairing (A/B runs): 0 auto (2-CTA clusters + dQ exchange), 1 single CTAs, 2 clusters without the exchange")
    ap.add_argument("--bwd-piece-blocks", type=int, default=0, help="plan desc field bwd_piece_blocks (A/B runs): Q blocks per tile_bwd work item, 0 = default")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            d = json.loads(p.read_text())
            return {k: float(d[k]) for k in FALLBACK_PEAKS}, "measured"
        except Exception:
            pass
    return dict(FALLBACK_PEAKS), "fallback"


# ------------------------------------------------------------------------------------------ clocks
CLOCK_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
               "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")


class ClockSampler:
    """nvidia-smi sampled every 200 ms DURING the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, device_index: int):
        self.proc = None
        self.idx = device_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={CLOCK_QUERY}", "--format=csv,noheader,nounits", "-lms", "200",
                                          "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for nm, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ oracle leg
def oracle_inputs_cpu(w):
    """Seeded host inputs for the oracle-only arm: the query heads of KV head 0's group (the oracle's cost per
    (row, head) does not depend on which head), generated on the CPU with the workload's recipe."""
    from dataclasses import replace

    import numpy as np
    import torch

    from paper_2512_20968_b200 import workloads as W

    g = w.heads_q // w.heads_kv
    ws = replace(w, heads_q=g, heads_kv=1)
    inp = W.make_inputs(ws, "cpu", ("q", "k", "v", "do") if w.backward else ("q", "k", "v"))
    return {k: t[0].contiguous().view(torch.int16).numpy().view(np.uint16) for k, t in inp.items()}


def oracle_inputs_from_device(w, inp):
    """Host copy (bf16 bits) of KV head 0 and its query-head group from the device inputs of the GPU arm."""
    import numpy as np
    import torch

    g = w.heads_q // w.heads_kv
    out = {}
    for k, t in inp.items():
        h = g if k in ("q", "do") else 1
        out[k] = t[0, :, :h, :].contiguous().cpu().view(torch.int16).numpy().view(np.uint16)
    return out


class OracleSample:
    """The oracle as it stands (oracle/attn_oracle.py, fp64, OpenMP over sampled rows) on a bounded sample of the
    workload: R random query rows of query head 0 -> forward (O, LSE from the definition), the query-side backward
    (LSE, Delta, dQ) and the key-side backward (dK, dV of KSAMPLE random keys, summed over those R rows).  Algorithmic FLOPs
    of the sample: 4*D per visible (q,k) pair forward, 6*D query side (the S, dP and dQ contractions), 4*D per visible pair
    of the (R rows x KSAMPLE keys) key-side sample (the dV and dK contractions): all 10*D of the backward are sampled."""

    KSAMPLE = 8192

    def __init__(self, w, host, seconds: float):
        import numpy as np

        from oracle import attn_oracle as oracle

        oracle.build()
        self.np, self.oracle, self.w, self.host = np, oracle, w, host
        self.threads = oracle.num_threads()
        self.pos = oracle.positions(w.n, w.L, w.seq_layout)
        self.rng = np.random.default_rng(20968)
        self.last = {}
        dt, _ = self.run(self.rows(self.threads))                      # calibration pass
        per_round = max(dt, 1e-3)
        self.R = int(max(1, min(4096, round(seconds / per_round)))) * self.threads

    def rows(self, count):
        return self.np.sort(self.rng.integers(0, self.w.seq_total, count)).astype(self.np.int64)

    def run(self, rows):
        np, w, h = self.np, self.w, self.host
        heads = np.zeros(len(rows), dtype=np.int32)
        D = w.head_dim
        t0 = time.perf_counter()
        self.oracle.fwd_rows(h["q"], h["k"], h["v"], w.scale, w.causal, self.pos, rows, heads)
        t1 = time.perf_counter()
        vis = int((self.pos[rows] + 1).sum()) if w.causal else len(rows) * w.seq_total
        flops = vis * D * 4.0
        part = {"rows": len(rows), "pairs_rows": vis, "s_fwd": t1 - t0, "s_dq": 0.0, "s_dkv_call": 0.0, "pairs_keys": 0}
        if w.backward:
            self.oracle.bwd_dq_rows(h["q"], h["k"], h["v"], h["do"], w.scale, w.causal, self.pos, rows, heads)
            t2 = time.perf_counter()
            keys = np.sort(self.rng.integers(0, w.seq_total, min(self.KSAMPLE, w.seq_total))).astype(np.int64)
            # query head 0 only: a one-head view keeps the key side at the sampled head (GQA: head 0 of KV head 0's group)
            q1, do1 = h["q"][:, :1], h["do"][:, :1]
            self.oracle.bwd_dkv_keys(q1, h["k"], h["v"], do1, w.scale, w.causal, self.pos, keys, np.zeros(len(keys), np.int32), qs_rows=rows)
            t3 = time.perf_counter()
            if w.causal:
                pk = np.sort(self.pos[keys])
                vis_k = int(np.searchsorted(pk, self.pos[rows], side="right").sum())     # keys of the sample each sampled row sees
            else:
                vis_k = len(rows) * len(keys)
            flops += vis * D * 6.0 + vis_k * D * 4.0
            part.update(s_dq=t2 - t1, s_dkv_call=t3 - t2, pairs_keys=vis_k)
        self.last = part
        return time.perf_counter() - t0, flops

    def timed(self):
        dt, flops = self.run(self.rows(self.R))
        return dt, flops

    def extrapolate(self):
        """Full-problem time of the oracle from the last sample: each leg scaled by (all visible pairs x all query heads) /
        (the pairs that leg sampled).  bwd_dkv_keys recomputes LSE and Delta of its query rows with bwd_dq_rows before its
        own loop (the oracle as it stands), so its call is split into that pass (it scales with the rows) and the key-side
        loop proper (it scales with the (row, key) pairs)."""
        w, p = self.w, self.last
        if not p or not p["pairs_rows"]:
            return {}
        all_pairs = float(w.visible_pairs()) * w.heads_q * w.batch
        per_row_legs = p["s_fwd"] + p["s_dq"] + (min(p["s_dq"], p["s_dkv_call"]) if w.backward else 0.0)
        sec = per_row_legs * all_pairs / p["pairs_rows"]
        if w.backward and p["pairs_keys"]:
            sec += max(p["s_dkv_call"] - p["s_dq"], 0.0) * all_pairs / p["pairs_keys"]
        fl = w.flops_fwd() + (w.flops_bwd() if w.backward else 0.0)
        return {"extrapolated_full_problem_seconds": sec, "extrapolated_tokens_per_s": w.seq_total * w.batch / sec,
                "extrapolated_tflops": fl / sec / 1e12, "sample_seconds": {k: p[k] for k in ("s_fwd", "s_dq", "s_dkv_call")},
                "sampled_pairs": {"query_rows_x_all_keys": p["pairs_rows"], "query_rows_x_sampled_keys": p["pairs_keys"]},
                "all_visible_pairs_x_heads": all_pairs}

    def describe(self):
        return (f"{self.R} random query rows of head 0 of {self.w.name}: fp64 forward rows"
                + (f" + query-side backward rows (dQ, Delta), all keys + key-side backward (dK, dV) of {min(self.KSAMPLE, self.w.seq_total)} random keys over those rows"
                   if self.w.backward else "") + "; all keys for the row legs")


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2512_20968_b200 import workloads as W

    w = W.CONFIGS[args.workload]
    host = oracle_inputs_cpu(w)
    smp = OracleSample(w, host, args.cpu_seconds)
    for _ in range(args.warmup):
        smp.run(smp.rows(smp.threads))                                  # warm-up: one row per thread
    tot_t = tot_f = 0.0
    for _ in range(args.steps):
        dt, fl = smp.timed()
        tot_t += dt
        tot_f += fl
    val = tot_f / tot_t / 1e12
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(1, args.steps), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, "oracle sample per step: " + smp.describe()),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": smp.threads, "kind": "oracle", "sample": smp.describe(), **smp.extrapolate()},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(w, note=""):
    cfg = {
        "workload": f"{w.name} (BASELINE.json configs[{w.index - 1}])", "mask": "causal" if w.causal else "non-causal",
        "mesh": f"{w.a}x{w.b}", "n": w.n, "seq_total": w.seq_total, "L": w.L, "batch": w.batch, "heads_q": w.heads_q,
        "heads_kv": w.heads_kv, "head_dim": w.head_dim, "seq_layout": w.seq_layout, "kvr": w.kvr, "order": w.order,
        "k_q": w.k_q, "k_kv": w.k_kv, "passes": "fwd+merge+bwd" if w.backward else "fwd+merge",
        "inputs": "bf16 iid N(0,1)" + (" with 4 of 128 Q/K channels x8" if w.outlier else ""),
        "precision": "split hi+lo P/dS operands (the mode parity-tested on outlier scores)" if w.outlier else "single bf16 operands",
        "l2": "inputs larger than L2 (no flush needed)" if w.seq_total * w.heads_q * w.head_dim * 2 > (126 << 20) else "L2-resident (report only)",
    }
    if note:
        cfg["note"] = note
    return cfg


# ------------------------------------------------------------------------------------------ multi-rank bookkeeping
def max_over_ranks(ms: float, dist, device) -> float:
    """Timing of the whole job = the slowest rank (replicas run independently)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch

    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tflops(flops_per_rank_step: float, world: int, steps: int, ms_total: float) -> float:
    """value = units all ranks processed / max-over-ranks time (weak scaling: every rank runs the full workload)."""
    return world * flops_per_rank_step * steps / (ms_total / 1e3) / 1e12


# ------------------------------------------------------------------------------------------ GPU arm
def physical_gpu_index(local_rank: int) -> int:
    """nvidia-smi index of this rank's GPU (CUDA_VISIBLE_DEVICES may renumber them)."""
    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
    ids = [x for x in vis.split(",") if x.strip()]
    if local_rank < len(ids) and ids[local_rank].strip().isdigit():
        return int(ids[local_rank])
    return local_rank


def alloc_host(shape, dtype, torch):
    """pinned host buffer; pageable if the box refuses to pin that much"""
    try:
        return torch.empty(shape, dtype=dtype, pin_memory=True), True
    except RuntimeError:
        return torch.empty(shape, dtype=dtype), False


def run_e2e(plan, w, inp, buf, torch, steps):
    """The public host-buffer call (mesh_attn_step_host): H2D of Q,K,V(,dO), the whole hot path, D2H of O, LSE
    (and dQ,dK,dV), all inside the timed region.  The device staging buffers are SEPARATE from the resident inputs and
    NaN-filled before every timed call, so the kernels can only have seen what the timed copies brought; afterwards the O that
    came back to the host is compared bit for bit with a device-resident forward on the original inputs (the forward has no
    atomics: same bits), which proves the copy -> kernel -> copy chain of the timed call."""
    host_in, host_out, stage, pinned = {}, {}, {}, True
    for k, t in inp.items():
        host_in[k], p = alloc_host(t.shape, t.dtype, torch)
        pinned &= p
        host_in[k].copy_(t)
        stage[k] = torch.empty_like(t)
    outs = {"O": buf.O, "lse": buf.lse}
    if w.backward:
        outs.update(dQ=buf.dQ, dK=buf.dK, dV=buf.dV)
    for k, t in outs.items():
        host_out[k], p = alloc_host(t.shape, t.dtype, torch)
        pinned &= p
        host_out[k].zero_()                                   # touch the pages before timing
    kw = dict(Q_host=host_in["q"], K_host=host_in["k"], V_host=host_in["v"], O_host=host_out["O"], lse_host=host_out["lse"],
              d_Q=stage["q"], d_K=stage["k"], d_V=stage["v"], d_O=buf.O, d_lse=buf.lse, d_partial_O=buf.partial_O,
              d_partial_lse=buf.partial_lse)
    if w.backward:
        kw.update(dO_host=host_in["do"], dQ_host=host_out["dQ"], dK_host=host_out["dK"], dV_host=host_out["dV"], d_dO=stage["do"],
                  d_bwd_ws=buf.bwd_ws, d_dQ=buf.dQ, d_dK=buf.dK, d_dV=buf.dV)
    ms = 0.0
    for _ in range(steps):
        for t in stage.values():
            t.view(torch.int16).fill_(0x7FC0)                 # bf16 NaN: nothing of the resident inputs survives in the staging
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        plan.step_host(**kw)                                  # synchronises its stream before returning
        e1.record()
        torch.cuda.synchronize()
        ms += e0.elapsed_time(e1)
    ms /= steps
    h2d = sum(t.numel() * t.element_size() for t in host_in.values())
    d2h = sum(t.numel() * t.element_size() for t in host_out.values())
    # ---- check: the staging now holds the inputs, and the host O equals a resident forward's O
    checked = all(torch.equal(stage[k].view(torch.int16), inp[k].view(torch.int16)) for k in inp)
    del stage
    plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
    torch.cuda.synchronize()
    rows = 1 << 15
    for r0 in range(0, w.seq_total, rows):
        r1 = min(w.seq_total, r0 + rows)
        checked = checked and bool(torch.equal(host_out["O"][:, r0:r1].cuda(), buf.O[:, r0:r1]))
    if w.backward:                                            # atomics reorder the gradient sums: finite and non-trivial is what can be said
        checked = checked and all(bool(torch.isfinite(host_out[k][:, :rows]).all().item()) and bool(host_out[k][:, :rows].abs().max().item() > 0)
                                  for k in ("dQ", "dK", "dV"))
    return ms, h2d, d2h, pinned, checked


def run_ours(args):
    import torch

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    import __graft_entry__ as entry

    if rank == 0:
        import contextlib

        with contextlib.redirect_stdout(sys.stderr):
            entry.build()
    if dist is not None:
        dist.barrier()
    from paper_2512_20968_b200 import Buffers, launch_count, plan_for
    from paper_2512_20968_b200 import binding as B
    from paper_2512_20968_b200 import workloads as W

    w = W.CONFIGS[args.workload]
    peaks, peak_src = load_peaks()
    inp = W.make_inputs(w, "cuda", ("q", "k", "v", "do") if w.backward else ("q", "k", "v"))
    plan = plan_for(w, usp_lanes=args.usp_lanes, bwd_pairing=args.bwd_pairing, bwd_piece_blocks=args.bwd_piece_blocks, fwd_pairing=args.fwd_pairing)
    buf = Buffers(plan, w, backward=w.backward)

    def step():
        plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse)
        if w.backward:
            plan.backward(inp["q"], inp["k"], inp["v"], buf.O, inp["do"], buf.lse, buf.bwd_ws, buf.dQ, buf.dK, buf.dV)

    def fence():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    fence()
    clocks = ClockSampler(physical_gpu_index(local_rank))
    if rank == 0:
        clocks.start()
    B.profile_enable(True, 8192)
    n0 = launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    fence()
    ms_total = e0.elapsed_time(e1)
    launches = launch_count() - n0
    clk = clocks.stop() if rank == 0 else None
    prof = {name: B.profile_read(kind) for name, kind in (("tile_fwd", B.K_TILE_FWD), ("merge", B.K_MERGE),
                                                          ("bwd_preprocess", B.K_BWD_PREPROCESS), ("tile_bwd", B.K_TILE_BWD))}
    B.profile_enable(False)
    ms_total = max_over_ranks(ms_total, dist, "cuda")

    K = args.steps
    fl_fwd, fl_bwd = plan.query(B.Q_FLOPS_FWD), (plan.query(B.Q_FLOPS_BWD) if w.backward else 0)
    sec = ms_total / 1e3
    value = whole_job_tflops(fl_fwd + fl_bwd, world, K, ms_total)

    e2e = None
    if not args.no_e2e:
        try:
            e2e_steps = 1 if ms_total / K > 2000 else min(K, 5)
            ms_e, h2d, d2h, pinned, checked = run_e2e(plan, w, inp, buf, torch, e2e_steps)
            ms_e = max_over_ranks(ms_e, dist, "cuda")
            e2e = {"value": whole_job_tflops(fl_fwd + fl_bwd, world, 1, ms_e), "unit": UNIT, "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": d2h, "ms_per_step": ms_e, "steps": e2e_steps, "pinned": pinned,
                   "api": "mesh_attn_step_host", "checked": checked,
                   "check": "device staging separate from the resident inputs and NaN-filled before the timed call; afterwards staging == inputs "
                            "and the host O == a resident forward's O bit for bit; host gradients finite and non-zero"}
        except (RuntimeError, MemoryError) as ex:                # host or device memory too small for the mirrors / the staging
            e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "error": str(ex)[:200]}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel, per launch, from the events recorded inside the timed region
    dom = max(("tile_fwd", "tile_bwd"), key=lambda k: prof[k][0])
    dom_ms, dom_n = prof[dom]
    dom_flops = (fl_fwd if dom == "tile_fwd" else fl_bwd) * K            # all launches of the timed region together
    long_step = sec >= 2.0
    peak = peaks["bf16_tflops_sustained"] if long_step else peaks["bf16_tflops"]
    ach = dom_flops / (dom_ms / 1e3) / 1e12 if dom_ms > 0 else 0.0
    traffic, traffic_src = load_traffic(w.name, dom)
    roofline = {"kernel": f"mesh_attn_{dom}", "bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": ach / peak, "traffic": traffic, "traffic_source": traffic_src, "launches": dom_n, "avg_launch_ms": dom_ms / max(1, dom_n),
                "algorithmic_flops_per_launch": dom_flops / max(1, dom_n),
                "peak_kind": f"{peak_src} dense bf16, " + ("sustained (kernel timed inside a long step)" if long_step else "burst"),
                "share_of_step": dom_ms / ms_total}
    kernels = {}
    for name, (ms, n) in prof.items():
        if n:
            kernels[name] = {"launches": n, "ms_total": ms, "share_of_step": ms / ms_total}
    if prof["tile_fwd"][0] > 0:
        kernels["tile_fwd"]["tflops"] = fl_fwd * K / (prof["tile_fwd"][0] / 1e3) / 1e12
        kernels["tile_fwd"]["frac_of_peak"] = kernels["tile_fwd"]["tflops"] / peak
    if prof["tile_bwd"][0] > 0:
        kernels["tile_bwd"]["tflops"] = fl_bwd * K / (prof["tile_bwd"][0] / 1e3) / 1e12
        kernels["tile_bwd"]["frac_of_peak"] = kernels["tile_bwd"]["tflops"] / peak
    if prof["merge"][0] > 0:
        mbytes = plan.query(B.Q_MERGE_BYTES) * prof["merge"][1]
        kernels["merge"]["gbs"] = mbytes / (prof["merge"][0] / 1e3) / 1e9
        kernels["merge"]["frac_of_hbm"] = kernels["merge"]["gbs"] / peaks["hbm_gbs"]
    fwd_ms = prof["tile_fwd"][0] + prof["merge"][0]
    summary = {"fwd_tflops_incl_merge": fl_fwd * K / (fwd_ms / 1e3) / 1e12 if fwd_ms > 0 else None,
               "fwd_bwd_tflops": value / world,
               "pct_of_bf16_peak": {"measured_burst": 100 * value / world / peaks["bf16_tflops"],
                                    "measured_sustained": 100 * value / world / peaks["bf16_tflops_sustained"],
                                    "nominal_2250": 100 * value / world / 2250.0}}

    cpu = None
    if not args.no_cpu_baseline:
        smp = OracleSample(w, oracle_inputs_from_device(w, inp), args.cpu_seconds)
        dt, fl = smp.timed()
        cpu = {"value": fl / dt / 1e12, "unit": UNIT, "cores": smp.threads, "kind": "oracle", "sample": smp.describe(),
               "seconds": dt, **smp.extrapolate()}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
        "data": "synthetic", "config": workload_config(w, "N>1: independent replicas, no collective (DESIGN.md)" if world > 1 else ""),
        "clocks": clk, "e2e": e2e, "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu, "kernels": kernels,
        "summary": summary,
    }
    if args.usp_lanes > 1:
        line["config"]["usp_lanes"] = args.usp_lanes
    line["config"]["tile_fwd_kernel"] = {0: "single CTAs", 1: "2-CTA clusters, tcgen05 cta_group::2 MMAs (K / V halves per CTA)"}[plan.query(B.Q_FWD_PAIRED)]
    line["config"]["tile_bwd_kernel"] = {0: "single CTAs", 1: "2-CTA clusters, shared Q/dO tile loads", 2: "2-CTA clusters, shared tile loads + dQ exchange"}[plan.query(B.Q_BWD_PAIRED)]
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_goo_executor(args):
    """the forward step list executed task by task.  Prints one JSON line of its own."""
    import torch

    import __graft_entry__ as entry
    import contextlib
    with contextlib.redirect_stdout(sys.stderr):
        entry.build()
    from paper_2512_20968_b200 import Buffers, plan_for
    from paper_2512_20968_b200 import binding as B
    from paper_2512_20968_b200 import workloads as W

    torch.cuda.set_device(0)
    w = W.CONFIGS[args.workload]
    inp = W.make_inputs(w, "cuda", ("q", "k", "v"))
    plan = plan_for(w)
    buf = Buffers(plan, w, backward=False)
    f32 = dict(dtype=torch.float32, device="cuda")
    part_O = torch.empty(plan.query(B.Q_GOO_PARTIAL_O_BYTES) * w.a // 4, **f32)
    part_lse = torch.empty(plan.query(B.Q_GOO_PARTIAL_LSE_BYTES) * w.a // 4, **f32)
    comm_ws = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def timed(fn):
        best = []
        for it in range(args.warmup + args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            if it >= args.warmup:
                best.append(e0.elapsed_time(e1))
        return statistics.median(best)

    R = args.goo_executor
    goo = lambda rep, ov: [plan.forward_goo(r, inp["q"], inp["k"], inp["v"], buf.O, buf.lse, part_O, part_lse, comm_ws=comm_ws,
                                            comm_repeat=rep, overlap=ov) for r in range(w.b)]
    t_fused = timed(lambda: plan.forward(inp["q"], inp["k"], inp["v"], buf.O, buf.lse, buf.partial_O, buf.partial_lse))
    t_compute = timed(lambda: goo(0, True))
    t_overlap = timed(lambda: goo(R, True))
    t_serial = timed(lambda: goo(R, False))
    makespan, serial, exposed = plan.timeline()
    steps = plan.steps()
    line = {
        "mode": "goo_executor", "config": workload_config(w), "comm_repeat": R,
        "comm_bytes_per_q_group": plan.query(B.Q_GOO_COMM_BYTES), "steps": int(steps[:, 0].max()) if len(steps) else 0,   # step numbers are 1-based
        "compute_tasks_per_q_group": w.k_q * w.k_kv,
        "ms": {"fused_forward": t_fused, "executor_no_comm": t_compute, "executor_overlapped": t_overlap, "executor_serialised": t_serial},
        "exposed_comm_ms": {"overlapped": t_overlap - t_compute, "serialised": t_serial - t_compute},
        "model_cost_units": {"makespan": makespan, "serial": serial, "exposed_comm": exposed},
    }
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.goo_executor >= 0:
        run_goo_executor(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
