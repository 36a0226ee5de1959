"""Pins of oracle/plan_oracle.py against the values the paper prints
(tests/golden/paper_planner_examples.txt) and structural invariants."""
from pathlib import Path

import pytest

from oracle import plan_oracle as po

GOLD = {}
for line in (Path(__file__).parent / "golden" / "paper_planner_examples.txt").read_text().splitlines():
    line = line.split("#")[0].strip()
    if "=" in line:
        k, v = (x.strip() for x in line.split("="))
        GOLD[k] = v


def ints(key):
    return [int(x) for x in GOLD[key].split(",")]


def test_fig1_units():
    ring, basic, kvr = po.ring_matrix(9), po.assignment_matrix(9, 3, 3, False), po.assignment_matrix(9, 3, 3, True)
    assert po.comm_units(ring) == int(GOLD["ring_units_total_n9"])
    assert po.comm_units(basic) == int(GOLD["basic_units_total_n9"])
    assert po.comm_units(kvr) == int(GOLD["kvr_units_total_n9"])
    for g in range(9):
        _, _, RQ, RKV = po.footprints(ring, g)
        assert len(RQ) + 2 * len(RKV) == int(GOLD["ring_units_per_gpu_n9"])
        _, _, RQ, RKV = po.footprints(basic, g)
        want = GOLD["basic_units_diag_gpu_n9"] if g in (0, 4, 8) else GOLD["basic_units_offdiag_gpu_n9"]
        assert len(RQ) + 2 * len(RKV) == int(want)


def test_fig1_footprints_gpu3():
    IQ, IKV, RQ, RKV = po.footprints(po.assignment_matrix(9, 3, 3, False), 3)
    assert (IQ, IKV, RQ, RKV) == (ints("basic_gpu3_IQ"), ints("basic_gpu3_IKV"), ints("basic_gpu3_RQ"), ints("basic_gpu3_RKV"))
    assert len(RQ) + len(RKV) == int(GOLD["basic_gpu3_remote_total"])
    IQ, IKV, RQ, RKV = po.footprints(po.assignment_matrix(9, 3, 3, True), 3)
    assert IKV == ints("kvr_gpu3_IKV") and RKV == ints("kvr_gpu3_RKV")
    # KV order after rotation = concatenation of the tile columns' footprints
    order = [j for c in range(3) for j in po.footprints(po.assignment_matrix(9, 3, 3, True), c)[1]]
    assert order == ints("kvr_kv_order_n9")


def test_fig3_groups():
    assert po.q_group(0, 3) == ints("a3b5_gpu0_qgroup")
    assert po.kv_group(0, 3, 5) == ints("a3b5_gpu0_kvgroup")
    A = po.assignment_matrix(15, 3, 5, True)
    assert po.footprints(A, 0)[1] == ints("a3b5_gpu0_kvgroup")
    assert po.footprints(A, 1)[1] == ints("a3b5_gpu1_kv")
    assert po.footprints(A, 2)[1] == ints("a3b5_gpu2_kv")


@pytest.mark.parametrize("a,b", [(1, 4), (4, 1), (2, 2), (3, 3), (3, 5), (5, 3), (4, 4), (8, 8), (16, 16), (8, 32)])
def test_structural_invariants(a, b):
    n = a * b
    for kvr in (False, True):
        A = po.assignment_matrix(n, a, b, kvr)
        flat = [g for row in A for g in row]
        assert all(flat.count(g) == n for g in range(n))          # every GPU gets exactly n cells (L116)
        for g in range(n):
            IQ, IKV, RQ, RKV = po.footprints(A, g)
            assert len(IQ) == a and len(IKV) == b
            assert g in IQ and len(RQ) == a - 1                    # L133
            if kvr:
                assert g in IKV and len(RKV) == b - 1              # L161
                assert IKV == po.kv_group(g % a, a, b)             # the KV group owns its footprint (L161)
            else:
                assert len(RKV) in (b - 1, b)                      # L133
            assert IQ == po.q_group(g // a, a)
        if a == b:
            assert max(len(po.footprints(A, g)[2]) + len(po.footprints(A, g)[3]) for g in range(n)) <= 2 * a - 1  # L137
    # groups partition 0..n-1 (L178-182)
    assert sorted(x for r in range(b) for x in po.q_group(r, a)) == list(range(n))
    assert sorted(x for c in range(a) for x in po.kv_group(c, a, b)) == list(range(n))


def test_tam_example():
    q, kv = po.tam_internode_units(8, 8, 8, 8)
    assert q == 0 and q + kv == int(GOLD["tam_alpha8_node0_units"])
    q, kv = po.tam_internode_units(8, 8, 8, 4)
    assert (q, kv, q + kv) == (int(GOLD["tam_alpha4_node0_q_units"]), int(GOLD["tam_alpha4_node0_kv_units"]),
                               int(GOLD["tam_alpha4_node0_units"]))


def test_volume_closed_forms():
    gib = 2.0 ** 30
    Nd = 524288 * 8192                      # 512K tokens, hidden 8192
    assert round(po.mesh_volume_fwd(16, 16, Nd) * 2 / gib, 1) == float(GOLD["mesh_16x16_fwd_gib"])
    assert round(2 * po.mesh_volume_fwd(16, 16, Nd) * 2 / gib, 1) == float(GOLD["mesh_16x16_bwd_gib"])
    assert round(po.ring_volume_fwd(256, Nd) * 2 / gib, 1) == float(GOLD["ring_fwd_gib"])
    assert round(2 * po.ring_volume_fwd(256, Nd) * 2 / gib, 1) == float(GOLD["ring_bwd_gib"])
    assert round(po.ring_volume_fwd(256, 1048576 * 8192) * 2 / gib) == int(GOLD["ring_kv_per_gpu_1m_gib"])
    # the closed form equals the footprint count: |R^Q| (Q in) + |R^Q| (O out) + 2|R^KV|, one unit = Nd/n
    for a, b in [(3, 3), (3, 5), (16, 16)]:
        A = po.assignment_matrix(a * b, a, b, True)
        _, _, RQ, RKV = po.footprints(A, 0)
        assert (2 * len(RQ) + 2 * len(RKV)) / (a * b) == pytest.approx(po.mesh_volume_fwd(a, b, 1.0))


def test_goo_fig4_example():
    steps = po.goo_forward(3, 3, t_ag_kv=1.0, t_ag_q=0.5, t_rs_q=0.5, t_c=0.5, gamma=1.0)
    name = {po.AG_KV: "AGKV", po.AG_Q: "AGQ", po.RS_Q: "RSQ"}
    comm = [None if c is None else f"{name[c[0]]}{c[1]}" for c, _ in steps]
    assert comm[:6] == GOLD["goo_comm_steps_1_to_6"].split(",")
    assert [f"C{i}{j}" for i, j in steps[2][1]] == GOLD["goo_step3_compute"].split(",")
    assert [f"C{i}{j}" for i, j in steps[5][1]] == GOLD["goo_step6_compute"].split(",")
    assert [k + 1 for k, (c, _) in enumerate(steps) if c is None] == ints("goo_compute_only_steps")
    assert sum(c is not None for c, _ in steps) == int(GOLD["goo_num_comm_steps"])


@pytest.mark.parametrize("kq,kkv", [(1, 1), (2, 2), (4, 4), (1, 16), (16, 1), (3, 5), (2, 8)])
def test_goo_validity(kq, kkv):
    for costs in [(1.0, 0.5, 0.5, 0.5), (0.3, 0.7, 0.2, 1.0), (2.0, 2.0, 2.0, 0.1)]:
        steps = po.goo_forward(kq, kkv, *costs, gamma=1.05)
        seen_kv, seen_q, seen_rs, done_c = set(), set(), set(), set()
        for comm, fill in steps:
            for (i, j) in fill:                       # ready at the step boundary (L210)
                assert i in seen_q and j in seen_kv and (i, j) not in done_c
            if comm is not None:
                kind, idx = comm
                if kind == po.RS_Q:
                    assert all((idx, j) in done_c for j in range(kkv))   # L208
                    seen_rs.add(idx)
                elif kind == po.AG_Q:
                    seen_q.add(idx)
                else:
                    seen_kv.add(idx)
            else:
                assert len(fill) == 1                  # compute-only step has one task (L230)
            done_c.update(fill)
        assert len(done_c) == kq * kkv and len(seen_rs) == kq
        assert sum(c is not None for c, _ in steps) == 2 * kq + kkv
