"""C++ planner (through the C ABI, host only) against oracle/plan_oracle.py, the paper's printed
examples and structural invariants.  No GPU needed."""
from pathlib import Path

import numpy as np
import pytest

from oracle import plan_oracle as po
from paper_2512_20968_b200 import binding as B
from paper_2512_20968_b200.binding import MeshAttnError, Plan


def mk(a, b, L=128, **kw):
    base = dict(a=a, b=b, batch=1, seq_total=a * b * L, heads_q=2, heads_kv=1, head_dim=64)
    base.update(kw)
    return Plan(**base)


def test_library_exports_every_declared_symbol():
    import re
    from pathlib import Path

    header = (Path(__file__).parent.parent / "include" / "mesh_attn.h").read_text()
    code = re.sub(r"/\*.*?\*/", "", header, flags=re.S)          # declarations only, comments stripped
    declared = set(re.findall(r"\b(mesh_attn_[a-z_]+)\s*\(", code))
    assert declared == set(B.EXPORTED)
    for name in declared:
        assert hasattr(B.lib, name), name


@pytest.mark.parametrize("a,b", [(2, 2), (3, 3), (3, 5), (5, 3), (4, 4), (1, 4), (4, 1), (8, 8), (16, 16)])
@pytest.mark.parametrize("kvr", [0, 1])
def test_am_and_footprints_match_oracle(a, b, kvr):
    n = a * b
    p = mk(a, b, kvr=kvr)
    A = po.assignment_matrix(n, a, b, bool(kvr))
    assert p.am().tolist() == A
    for g in range(n):
        IQ, IKV, _, _ = po.footprints(A, g)
        iq, ikv = p.footprint(g)
        assert iq.tolist() == IQ and ikv.tolist() == IKV
    assert p.query(B.Q_COMM_UNITS) == po.comm_units(A)
    assert p.query(B.Q_WAVES) == b and p.query(B.Q_HAS_DEVICE) in (0, 1)


def test_paper_fig1_units():
    assert mk(3, 3, kvr=0).query(B.Q_COMM_UNITS) == 84
    assert mk(3, 3, kvr=1).query(B.Q_COMM_UNITS) == 72
    assert mk(3, 3, kvr=1).footprint(3)[1].tolist() == [0, 3, 6]


def _steps_to_oracle_form(rows):
    out = {}
    for step, kind, i, j in rows.tolist():
        comm, fill = out.setdefault(step, [None, []])
        if kind == B.TASK_C:
            fill.append((i, j))
        else:
            out[step][0] = (kind, j if kind in (B.TASK_AG_KV, B.TASK_RS_KV) else i)
    return [(tuple(v[0]) if v[0] else None, v[1]) for _, v in sorted(out.items())]


def test_goo_fig4_example():
    # k_Q = k_KV = 3, T = (AG-KV 1, AG-Q .5, RS-Q .5, C .5), gamma = 1
    p = mk(2, 2, L=384, order=1, k_q=3, k_kv=3, gamma=1.0, t_ag_kv=1.0, t_ag_q=0.5, t_rs_q=0.5, t_c=0.5)
    steps = _steps_to_oracle_form(p.steps())
    assert steps == po.goo_forward(3, 3, 1.0, 0.5, 0.5, 0.5, gamma=1.0)
    comm = [c for c, _ in steps]
    assert comm[:6] == [(B.TASK_AG_KV, 0), (B.TASK_AG_Q, 0), (B.TASK_AG_Q, 1), (B.TASK_AG_KV, 1), (B.TASK_AG_Q, 2), (B.TASK_AG_KV, 2)]
    assert steps[2][1] == [(0, 0)] and steps[5][1] == [(1, 1), (2, 0)]
    assert [k + 1 for k, c in enumerate(comm) if c is None] == [7, 10] and len(steps) == 11
    # timeline of that printed schedule, by hand: steps last 1, .5, .5, 1, .5, 1 (AG-KV-2 || C-1-1 + C-2-0), .5, .5, .5, .5, .5
    makespan, serial, exposed = p.timeline()
    assert (makespan, serial, exposed) == (7.0, 3 * 1.0 + 6 * 0.5 + 9 * 0.5, 7.0 - 9 * 0.5)
    # row-major order has a single step: all communication first, nothing hidden
    q = mk(2, 2, L=384, order=0, k_q=3, k_kv=3, t_ag_kv=1.0, t_ag_q=0.5, t_rs_q=0.5, t_c=0.5)
    m2, s2, e2 = q.timeline()
    assert s2 == serial and m2 >= makespan and e2 >= exposed


def _assert_same_tiles(got, ref, order):
    """What the paper fixes about a GPU's tile list: the SEQUENCE of compute tasks C-i-j (the step list)
    and, inside a task, the SET of pairs "for each gathered pair (Q_u, KV_v)" (Alg.2 l.3-5, L171-173) = I_g^Q x I_g^KV.
    The order of the pairs inside one task is a free choice (any order gives the same attention; reading R17),
    so it is compared as a set, not as a sequence."""
    got = [tuple(r) for r in got.tolist()]
    per = len(got) // len(order)
    assert len(got) == len(ref) == per * len(order)
    for t, ij in enumerate(order):
        g_chunk, r_chunk = got[t * per:(t + 1) * per], ref[t * per:(t + 1) * per]
        assert all(x[2:] == tuple(ij) for x in g_chunk)
        assert len(set(g_chunk)) == per and set(g_chunk) == set(r_chunk)


def test_tile_set_of_the_papers_example():
    # PAPER.md L141 + L161: n = 9, a = b = 3, GPU 3: I^Q = {3,4,5}; KV footprint {0,1,2} (basic) / {0,3,6} (KVR)
    for kvr, ikv in ((0, {0, 1, 2}), (1, {0, 3, 6})):
        t = mk(3, 3, L=128, kvr=kvr).tiles(3)
        assert {(int(u), int(v)) for u, v, _, _ in t.tolist()} == {(u, v) for u in (3, 4, 5) for v in ikv}
        assert {(u, v) for u, v, _, _ in po.tile_list(9, 3, 3, bool(kvr), 3, [(0, 0)])} == {(u, v) for u in (3, 4, 5) for v in ikv}


@pytest.mark.parametrize("kq,kkv", [(1, 1), (2, 2), (4, 4), (2, 8), (8, 2), (1, 16), (16, 1), (3, 5)])
@pytest.mark.parametrize("costs", [(1.0, 0.5, 0.5, 0.5), (0.3, 0.7, 0.2, 1.0), (2.0, 2.0, 2.0, 0.1)])
def test_goo_matches_oracle_and_tile_lists(kq, kkv, costs):
    L = 128 * kq * kkv
    p = mk(2, 3, L=L, kvr=1, order=1, k_q=kq, k_kv=kkv, t_ag_kv=costs[0], t_ag_q=costs[1], t_rs_q=costs[2], t_c=costs[3])
    ref = po.goo_forward(kq, kkv, *costs, gamma=1.05)
    assert _steps_to_oracle_form(p.steps()) == ref
    # timeline invariants: never longer than serial execution, never shorter than either lane alone
    makespan, serial, exposed = p.timeline()
    comm_total = kkv * costs[0] + kq * costs[1] + kq * costs[2]
    assert max(comm_total, kq * kkv * costs[3]) - 1e-9 <= makespan <= serial + 1e-9
    assert abs(serial - (comm_total + kq * kkv * costs[3])) < 1e-6 and abs(exposed - (makespan - kq * kkv * costs[3])) < 1e-6
    order = po.compute_order(ref)
    for g in range(6):
        _assert_same_tiles(p.tiles(g), po.tile_list(6, 2, 3, True, g, order), order)


def test_backward_goo_is_valid():
    # PAPER.md L238 omits the backward schedule: validity invariants only (parity unpinned)
    p = mk(2, 2, L=512, order=1, k_q=2, k_kv=2)
    rows = p.steps(backward=True).tolist()
    have_q, have_kv, done = set(), set(), set()
    for step in sorted({r[0] for r in rows}):
        cur = [r for r in rows if r[0] == step]
        for _, kind, i, j in cur:
            if kind == B.TASK_C:
                assert i in have_q and j in have_kv and (i, j) not in done
        for _, kind, i, j in cur:
            if kind == B.TASK_RS_Q:
                assert all((i, jj) in done for jj in range(2))
            if kind == B.TASK_RS_KV:
                assert all((ii, j) in done for ii in range(2))
        for _, kind, i, j in cur:
            if kind == B.TASK_C:
                done.add((i, j))
            elif kind == B.TASK_AG_Q:
                have_q.add(i)
            elif kind == B.TASK_AG_KV:
                have_kv.add(j)
        assert sum(1 for r in cur if r[1] != B.TASK_C) <= 1
    assert len(done) == 4
    kinds = [r[1] for r in rows]
    assert kinds.count(B.TASK_RS_Q) == 2 and kinds.count(B.TASK_RS_KV) == 2


def test_row_major_order_and_queries():
    p = mk(3, 3, L=256, kvr=1, heads_q=4, heads_kv=2, head_dim=128, batch=2)
    t = p.tiles(4)
    _assert_same_tiles(t, po.tile_list(9, 3, 3, True, 4, [(0, 0)]), [(0, 0)])
    N = 9 * 256
    assert p.query(B.Q_FLOPS_FWD) == 4 * 128 * 4 * 2 * N * N
    assert p.query(B.Q_FLOPS_BWD) == 10 * 128 * 4 * 2 * N * N
    assert p.query(B.Q_SLOTS_PER_GPU) == 3
    assert p.query(B.Q_PARTIAL_O_BYTES) == 3 * 2 * 256 * 4 * 128 * 4
    assert p.query(B.Q_PARTIAL_LSE_BYTES) == 3 * 2 * 256 * 4 * 4
    assert p.query(B.Q_BLOCKS_FWD) == (N // 128) ** 2 * 4 * 2
    assert p.query(B.Q_FWD_ITEMS_PER_GPU) == 2 * 4 * 3 * 1           # batch x heads x a x (256/256)
    assert p.query(B.Q_BWD_ITEMS_PER_GPU) == 2 * 2 * 3 * 2           # batch x kv heads x b x (256/128)
    pc = mk(2, 2, L=256, causal=1, seq_layout=1)
    # striped causal: pairs v<=u are lower-triangular incl. diagonal (3 of 4 blocks at L=256), v>u strictly lower (3 of 4 too:
    # block (0,1) fully masked, diagonal blocks partially) -> every pair computes 3 blocks
    assert pc.query(B.Q_BLOCKS_FWD) == 16 * 3 * 2
    assert pc.query(B.Q_FLOPS_FWD) == 4 * 64 * 2 * (1024 * 1025 // 2)


@pytest.mark.parametrize("bad", [
    dict(n=5), dict(seq_total=1000), dict(seq_total=4 * 64), dict(heads_q=3, heads_kv=2), dict(head_dim=96),
    dict(k_q=5, k_kv=4), dict(k_q=3), dict(causal=2), dict(batch=0),
])
def test_invalid_geometry_is_rejected_at_plan_creation(bad):
    kw = dict(a=2, b=2, n=4, batch=1, seq_total=4 * 256, heads_q=2, heads_kv=1, head_dim=64)
    kw.update(bad)
    with pytest.raises(MeshAttnError) as e:
        Plan(**kw)
    assert e.value.status in (B.EINVAL, B.EUNSUPPORTED)


def test_compute_calls_fail_loudly_without_gpu():
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    p = mk(2, 2)
    with pytest.raises(MeshAttnError) as e:
        p.tile_fwd(0, 1, 16, 16, 16, 16, 16, stream=0)
    assert e.value.status == B.ECUDA


def test_planner_analytics_against_paper_numbers():
    """S8(f).1: closed-form per-GPU volumes (Table 1 / Table 5) and the topology-aware mapping traffic (Section 3.6),
    against the values the paper prints (tests/golden) and the independent planner oracle."""
    from oracle import plan_oracle as po

    gold = {}
    for line in (Path(__file__).parent / "golden" / "paper_planner_examples.txt").read_text().splitlines():
        if "=" in line and not line.startswith("#"):
            k, v = line.split("#")[0].split("=")
            gold[k.strip()] = v.strip()
    gib = 2.0 ** 30
    # 256 GPUs (16 x 16), 512K tokens, hidden 8192 = 64 heads x 128, BF16 (Table 5)
    p = B.Plan(a=16, b=16, batch=1, seq_total=524288, heads_q=64, heads_kv=64, head_dim=128)
    fwd, bwd, ring = (p.query(x) for x in (B.Q_MESH_COMM_BYTES_FWD, B.Q_MESH_COMM_BYTES_BWD, B.Q_RING_COMM_BYTES_FWD))
    assert round(fwd / gib, 1) == float(gold["mesh_16x16_fwd_gib"]) and round(bwd / gib, 1) == float(gold["mesh_16x16_bwd_gib"])
    assert round(ring / gib, 1) == float(gold["ring_fwd_gib"])
    assert fwd == int(po.mesh_volume_fwd(16, 16, 524288 * 8192) * 2)
    # 64 GPUs, a = b = 8, 8 GPUs per node: row-major mapping (alpha = 8) vs 4-wide node tiles
    p = B.Plan(a=8, b=8, batch=1, seq_total=8 * 8 * 128, heads_q=1, heads_kv=1, head_dim=128)
    q, kv = p.tam_units(8, 8)
    assert q == 0 and q + kv == int(gold["tam_alpha8_node0_units"])
    assert p.tam_units(8, 4) == (int(gold["tam_alpha4_node0_q_units"]), int(gold["tam_alpha4_node0_kv_units"]))
    for alpha in (1, 2, 4, 8):
        for node in range(8):
            assert p.tam_units(8, alpha, node) == po.tam_internode_units(8, 8, 8, alpha, node)
    with pytest.raises(B.MeshAttnError):
        p.tam_units(8, 3)


def test_usp_lanes_geometry_and_all_to_all_volume():
    """S8(f).3, Mesh-USP: U lanes, each Mesh-Attention over 1/U of the heads.  The partial
    workspace of a simulated GPU shrinks by U, the algorithmic work does not change, there are b*U waves; the
    Ulysses all-to-all volume reduces, for one mesh GPU (n = 1) and MHA, to Table 1's 4(U-1)/U^2 N d."""
    kw = dict(a=2, b=2, batch=1, seq_total=4 * 256, heads_q=16, heads_kv=8, head_dim=128, causal=1, seq_layout=1)
    base = Plan(**kw)
    for U in (2, 4, 8):
        p = Plan(usp_lanes=U, **kw)
        assert p.query(B.Q_USP_LANES) == U and base.query(B.Q_USP_LANES) == 1
        for what in (B.Q_PARTIAL_O_BYTES, B.Q_PARTIAL_LSE_BYTES, B.Q_MERGE_BYTES, B.Q_FWD_ITEMS_PER_GPU, B.Q_BWD_ITEMS_PER_GPU):
            assert p.query(what) * U == base.query(what), what
        for what in (B.Q_FLOPS_FWD, B.Q_FLOPS_BWD, B.Q_BLOCKS_FWD, B.Q_BWD_WS_BYTES, B.Q_SLOTS_PER_GPU, B.Q_COMM_UNITS):
            assert p.query(what) == base.query(what), what
        assert p.query(B.Q_WAVES) == U * base.query(B.Q_WAVES)
        assert np.array_equal(p.am(), base.am())                       # every lane uses the same a x b mesh
    with pytest.raises(MeshAttnError) as e:
        Plan(usp_lanes=3, **kw)                                         # 8 KV heads do not split into 3 lanes
    assert e.value.status == B.EINVAL
    assert base.query(B.Q_USP_A2A_BYTES_FWD) == 0
    # pure Ulysses = one mesh GPU per lane: 4 (U-1)/U^2 N d elements (Table 1), 2 bytes each
    N, H, D = 8 * 1024, 16, 128
    for U in (2, 8, 16):
        p = Plan(usp_lanes=U, a=1, b=1, batch=1, seq_total=N, heads_q=H, heads_kv=H, head_dim=D)
        assert p.query(B.Q_USP_A2A_BYTES_FWD) == 4 * (U - 1) * N * H * D * 2 // (U * U)
    # GQA: K and V move Hkv heads only; n mesh GPUs per lane hold N/(n U) tokens each
    p = Plan(usp_lanes=4, **kw)
    assert p.query(B.Q_USP_A2A_BYTES_FWD) == (4 * 256 // (4 * 4)) * 3 * (2 * 16 + 2 * 8) * 128 * 2 // 4


def test_backward_item_pairing_rule():
    """tile_bwd shares Q / dO tile loads between two CTAs only when items 2k, 2k+1 visit the same Q blocks: always for
    non-causal plans, for striped-causal plans (same key block of two KV partitions: the causal offset 0 / -1 does not
    move the first visible Q block), never when the item count is odd or the contiguous causal layout shifts the walks."""
    kw = dict(batch=1, heads_q=2, heads_kv=1, head_dim=128)
    # 2 = paired with the dQ exchange (bwd_pairing = 0, single-operand precision), 1 = paired, shared tile loads only, 0 = single CTAs
    assert Plan(a=2, b=2, seq_total=4 * 256, **kw).query(B.Q_BWD_PAIRED) == 2
    assert Plan(a=2, b=2, seq_total=4 * 256, causal=1, seq_layout=1, **kw).query(B.Q_BWD_PAIRED) == 2
    assert Plan(a=4, b=4, seq_total=16 * 256, causal=1, seq_layout=1, order=1, kvr=1, **kw).query(B.Q_BWD_PAIRED) == 2
    assert Plan(a=2, b=2, seq_total=4 * 256, causal=1, seq_layout=0, **kw).query(B.Q_BWD_PAIRED) == 0
    assert Plan(a=1, b=1, seq_total=128, **kw).query(B.Q_BWD_PAIRED) == 0          # a single item
    assert Plan(a=3, b=3, seq_total=9 * 128, causal=1, seq_layout=1, **kw).query(B.Q_BWD_PAIRED) == 0   # 3 partitions per key block
    assert Plan(a=3, b=3, seq_total=9 * 256, **kw).query(B.Q_BWD_PAIRED) == 2
    # the plan descriptor's switch (no environment variable): never / shared loads only; split precision never exchanges
    assert Plan(a=3, b=3, seq_total=9 * 256, bwd_pairing=1, **kw).query(B.Q_BWD_PAIRED) == 0
    assert Plan(a=3, b=3, seq_total=9 * 256, bwd_pairing=2, **kw).query(B.Q_BWD_PAIRED) == 1
    assert Plan(a=3, b=3, seq_total=9 * 256, precision=1, **kw).query(B.Q_BWD_PAIRED) == 1
    with pytest.raises(MeshAttnError):
        Plan(a=3, b=3, seq_total=9 * 256, bwd_pairing=3, **kw)


def test_segment_lists_do_not_grow_with_batch_and_are_bounded():
    """FwdItem / BwdItem::seglist are 16 bits: the lists are built once (not per batch index), and a plan that would
    need more than 32767 of them is refused instead of wrapping to a negative index."""
    kw = dict(heads_q=1, heads_kv=1, head_dim=64)
    small = Plan(a=2, b=2, seq_total=4 * 512, batch=1, k_q=4, k_kv=1, order=1, **kw)
    big = Plan(a=2, b=2, seq_total=4 * 512, batch=9000, k_q=4, k_kv=1, order=1, **kw)      # 36 004 lists before the fix
    assert big.query(B.Q_FWD_ITEMS_PER_GPU) == 9000 * small.query(B.Q_FWD_ITEMS_PER_GPU)
    assert big.query(B.Q_BWD_ITEMS_PER_GPU) == 9000 * small.query(B.Q_BWD_ITEMS_PER_GPU)
    with pytest.raises(MeshAttnError):                      # per-pair partials: k_q * b lists
        Plan(a=1, b=4096, seq_total=4096 * 2048, batch=1, k_q=16, k_kv=1, partial_mode=1, **kw)


def test_plan_health_on_a_host_only_plan():
    p = Plan(a=2, b=2, seq_total=4 * 128, batch=1, heads_q=1, heads_kv=1, head_dim=64)
    p.health()                                              # no device, no fault: OK


def test_goo_executor_volumes():
    """The bytes the executor's communication stand-ins move for one Q group are a x the per-GPU closed form
    2(a+b-2) N d / n, whatever the chunking; its partial workspace holds k_kv slots per Q partition."""
    for k_q, k_kv in ((1, 1), (2, 2), (4, 2)):
        p = Plan(a=4, b=2, batch=1, seq_total=8 * 1024, heads_q=8, heads_kv=8, head_dim=128, order=1, k_q=k_q, k_kv=k_kv)
        assert p.query(B.Q_GOO_COMM_BYTES) == 4 * p.query(B.Q_MESH_COMM_BYTES_FWD)
        assert p.query(B.Q_GOO_PARTIAL_O_BYTES) == k_kv * p.query(B.Q_PARTIAL_O_BYTES)
        assert p.query(B.Q_GOO_PARTIAL_LSE_BYTES) == k_kv * p.query(B.Q_PARTIAL_LSE_BYTES)


def test_out_dtype_field_is_validated_and_sizes_the_backward_workspace():
    """plan desc field out_dtype (include/mesh_attn.h): 0 fp32, 1 bf16 outputs; with 1 the backward workspace also holds the fp32
    accumulators of dQ, dK, dV (host-only plans answer the query too)."""
    kw = dict(a=2, b=2, n=4, batch=2, seq_total=2048, heads_q=8, heads_kv=2, head_dim=128, causal=1, seq_layout=1)
    p0, p1 = Plan(**kw), Plan(out_dtype=1, **kw)
    planes = 2 * 2 * 8 * 2048 * 4
    assert p0.query(B.Q_BWD_WS_BYTES) == planes
    assert p1.query(B.Q_BWD_WS_BYTES) == planes + 2 * 2048 * (8 + 2 * 2) * 128 * 4
    for what in (B.Q_PARTIAL_O_BYTES, B.Q_PARTIAL_LSE_BYTES, B.Q_FLOPS_FWD, B.Q_FLOPS_BWD, B.Q_BWD_ITEMS_PER_GPU):
        assert p0.query(what) == p1.query(what)
    for bad in (-1, 2):
        with pytest.raises(MeshAttnError) as e:
            Plan(out_dtype=bad, **kw)
        assert e.value.status == B.EINVAL


def test_forward_item_pairing_rule():
    """MESH_ATTN_Q_FWD_PAIRED (tile_fwd as CTA pairs, tcgen05 cta_group::2): items 2k, 2k+1 must stream the same K / V blocks on
    every simulated GPU -- true for non-causal and striped-causal plans with an even item count, false for the contiguous causal
    layout with a > 1 (the pair's Q partitions see different KV partitions); head_dim 128 and precision 0 only; fwd_pairing = 1
    turns it off.  BASELINE.json's configs: C2, C4, C5 pair, C3 (contiguous, precision 1) and C1 (head_dim 64) do not."""
    base = dict(a=2, b=2, n=4, batch=1, seq_total=4 * 512, heads_q=4, heads_kv=4, head_dim=128)
    assert Plan(causal=0, **base).query(B.Q_FWD_PAIRED) == 1
    assert Plan(causal=1, seq_layout=1, **base).query(B.Q_FWD_PAIRED) == 1
    assert Plan(causal=1, seq_layout=0, **base).query(B.Q_FWD_PAIRED) == 0
    assert Plan(causal=1, seq_layout=0, **dict(base, a=1, b=4, heads_q=8, heads_kv=2)).query(B.Q_FWD_PAIRED) == 1   # a = 1: pairs inside a GQA group
    assert Plan(causal=1, seq_layout=1, precision=1, **base).query(B.Q_FWD_PAIRED) == 0
    assert Plan(causal=1, seq_layout=1, fwd_pairing=1, **base).query(B.Q_FWD_PAIRED) == 0
    assert Plan(causal=0, **dict(base, head_dim=64)).query(B.Q_FWD_PAIRED) == 0
    for bad in (-1, 2):
        with pytest.raises(MeshAttnError):
            Plan(fwd_pairing=bad, **base)
    from paper_2512_20968_b200 import plan_for, workloads as W
    got = {name: plan_for(W.scaled_down(w, 512)).query(B.Q_FWD_PAIRED) for name, w in W.CONFIGS.items() if name != "C1"}
    assert got == {"C2": 1, "C3": 0, "C4": 1, "C5": 1}, got
    assert plan_for(W.scaled_down(W.C2, 256)).query(B.Q_FWD_PAIRED) == 0     # 3 items per KV head: a pair would straddle two heads


def test_kernel_variants_chosen_for_the_baseline_configs_at_full_size():
    """Which tile kernels BASELINE.json's configs run at FULL size (host-only plans, no GPU needed): the CTA-pair forward
    (MESH_ATTN_Q_FWD_PAIRED) and the paired backward with the dQ exchange (MESH_ATTN_Q_BWD_PAIRED = 2) on C2, C4, C5; on C3
    (contiguous causal layout, precision 1) the single-CTA forward and the paired backward without the exchange (1); C1 (head_dim 64)
    does not pair the forward and runs no backward."""
    from paper_2512_20968_b200 import plan_for, workloads as W

    fwd = {name: plan_for(w).query(B.Q_FWD_PAIRED) for name, w in W.CONFIGS.items()}
    assert fwd == {"C1": 0, "C2": 1, "C3": 0, "C4": 1, "C5": 1}, fwd
    bwd = {name: plan_for(w).query(B.Q_BWD_PAIRED) for name, w in W.CONFIGS.items() if name != "C1"}
    assert bwd == {"C2": 2, "C3": 1, "C4": 2, "C5": 2}, bwd


def test_random_geometry_draws_make_valid_plans_and_reach_every_kernel_variant():
    """The seeded draws of tests/test_gpu_random_geometries.py (host arithmetic only) are all accepted by the planner, agree with the
    plan oracle's assignment matrix, and between them reach both forward kernels, the single-CTA and the exchanging backward,
    head_dim 64, GQA, both causal layouts, both footprints, both orders with chunks, batch 2 and two USP lanes."""
    from paper_2512_20968_b200 import plan_for
    from tests.test_gpu_random_geometries import SEEDS, geometry

    seen = set()
    for seed in SEEDS:
        w, overrides = geometry(seed)
        plan = plan_for(w, **overrides)
        assert np.array_equal(plan.am(), np.asarray(po.assignment_matrix(w.n, w.a, w.b, w.kvr))), seed
        seen |= {("fwd_pair", plan.query(B.Q_FWD_PAIRED)), ("bwd_pair", plan.query(B.Q_BWD_PAIRED)), ("D", w.head_dim), ("gqa", w.heads_q > w.heads_kv),
                 ("layout", w.seq_layout if w.causal else "nc"), ("kvr", w.kvr), ("order", w.order), ("chunks", w.k_q * w.k_kv > 1),
                 ("batch", w.batch), ("lanes", overrides["usp_lanes"]), ("outlier", w.outlier), ("pieces", overrides["bwd_piece_blocks"] > 0),
                 ("per_pair", overrides["partial_mode"])}
    want = {("fwd_pair", 0), ("fwd_pair", 1), ("bwd_pair", 0), ("bwd_pair", 1), ("bwd_pair", 2), ("outlier", True), ("pieces", True), ("per_pair", 1), ("D", 64), ("D", 128), ("gqa", True), ("gqa", False),
            ("layout", "striped"), ("layout", "contiguous"), ("layout", "nc"), ("kvr", True), ("kvr", False), ("order", "greedy"),
            ("order", "row_major"), ("chunks", True), ("batch", 2), ("lanes", 2)}
    assert want <= seen, want - seen
