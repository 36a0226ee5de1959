"""Plain-Python oracle of the Mesh-Attention planner -- TEST INFRASTRUCTURE ONLY.

Follows the paper step by step, in its notation.  Never imports the product package.

  assignment matrix A, footprints I/R
  basic 2-D tiling
  KV partition rotation
  Q groups / KV groups
  communication units of an AM
  GOO step-based greedy scheduler               PAPER.md L194-230 (worked example L226-230)
  closed-form per-GPU volume (Table 1)
  topology-aware mapping traffic

Readings where the paper is silent (R9-R12):
  - candidates are the lowest-index unscheduled chunk of each collective type (L226);
    RS-Q-i is a candidate once every C-i-* has finished; its profit is 0;
  - ties: higher profit, then AG-KV < AG-Q < RS-Q, then lower chunk index
    (reproduces the choices of steps 1 and 4 of Fig. 4);
  - fill: tasks ready at the step boundary, in (i, j) order, added while the running
    total is below gamma * T_comm (L220-224);
  - compute-only step: the first ready task in (i, j) order (L230).
"""
from __future__ import annotations

AG_KV, AG_Q, RS_Q, C, RS_KV = 0, 1, 2, 3, 4


def assignment_matrix(n: int, a: int, b: int, kvr: bool):
    """A[i][j] = g  <=>  GPU g computes (Q_i, KV_j).  GPU g has tile row r = g // a and tile
    column c = g mod a; Q rows ra..(r+1)a-1; KV columns cb..(c+1)b-1 (basic) or {c + t a} (KVR)."""
    assert n == a * b
    A = [[-1] * n for _ in range(n)]
    for g in range(n):
        r, c = g // a, g % a
        kv = [c + t * a for t in range(b)] if kvr else list(range(c * b, (c + 1) * b))
        for i in range(r * a, (r + 1) * a):
            for j in kv:
                assert A[i][j] == -1
                A[i][j] = g
    return A


def ring_matrix(n: int):
    """Ring-Attention: row i -> GPU i."""
    return [[i] * n for i in range(n)]


def footprints(A, g: int):
    n = len(A)
    cells = [(i, j) for i in range(n) for j in range(n) if A[i][j] == g]
    IQ = sorted({i for i, _ in cells})
    IKV = sorted({j for _, j in cells})
    RQ = [i for i in IQ if i != g]
    RKV = [j for j in IKV if j != g]
    return IQ, IKV, RQ, RKV


def q_group(r: int, a: int):
    return [r * a + x for x in range(a)]


def kv_group(c: int, a: int, b: int):
    return [c + a * x for x in range(b)]


def comm_units(A):
    """Aggregate units: every remote Q (1) + its returned partial O (1) + every remote KV (2 = K and V)."""
    n = len(A)
    total = 0
    for g in range(n):
        _, _, RQ, RKV = footprints(A, g)
        total += len(RQ) + 2 * len(RKV) + len(RQ)
    return total


def mesh_volume_fwd(a: int, b: int, Nd: float) -> float:
    """Per-GPU forward volume 2(a+b-2) Nd / n in elements."""
    return 2.0 * (a + b - 2) * Nd / (a * b)


def ring_volume_fwd(n: int, Nd: float) -> float:
    """(2 - 2/n) Nd."""
    return (2.0 - 2.0 / n) * Nd


def tam_internode_units(a: int, b: int, gpus_per_node: int, alpha: int, node: int = 0):
    """Inter-node units of one node when an alpha-wide, (gpus_per_node/alpha)-tall tile of the
    logical mesh (rows = Q groups, columns = position inside the Q group) is mapped to each node
    (PAPER.md L259-263).  Returns (Q-dimension units, KV-dimension units)."""
    rows_per_node = gpus_per_node // alpha
    tiles_per_row = a // alpha

    def node_of(g):
        r, c = g // a, g % a
        return (r // rows_per_node) * tiles_per_row + c // alpha

    members = [g for g in range(a * b) if node_of(g) == node]
    q_units = kv_units = 0
    for r in sorted({g // a for g in members}):          # each Q group the node intersects
        remote = [x for x in q_group(r, a) if node_of(x) != node]
        q_units += 2 * len(remote)                       # remote Q in + partial O out
    for c in sorted({g % a for g in members}):           # each KV group the node intersects
        remote = [x for x in kv_group(c, a, b) if node_of(x) != node]
        kv_units += 2 * len(remote)                      # K and V
    return q_units, kv_units


def goo_forward(k_q: int, k_kv: int, t_ag_kv: float, t_ag_q: float, t_rs_q: float, t_c: float, gamma: float = 1.05):
    """Step list [(comm or None, [compute tasks])], comm = (kind, idx), compute = (i, j)."""
    kv_next = q_next = 0                  # lowest-index unscheduled AG chunk of each type
    kv_done, q_done = set(), set()        # completed (scheduled in an EARLIER step)
    c_done, rs_done = set(), set()
    steps = []
    all_c = [(i, j) for i in range(k_q) for j in range(k_kv)]
    while len(rs_done) < k_q or len(c_done) < len(all_c):
        ready = [t for t in all_c if t not in c_done and t[0] in q_done and t[1] in kv_done]
        cands = []
        if kv_next < k_kv:
            unlock = sum(1 for i in q_done if (i, kv_next) not in c_done) * t_c
            cands.append((-(unlock / t_ag_kv), AG_KV, kv_next, t_ag_kv))
        if q_next < k_q:
            unlock = sum(1 for j in kv_done if (q_next, j) not in c_done) * t_c
            cands.append((-(unlock / t_ag_q), AG_Q, q_next, t_ag_q))
        for i in range(k_q):
            if i not in rs_done and all((i, j) in c_done for j in range(k_kv)):
                cands.append((0.0, RS_Q, i, t_rs_q))
                break
        if not cands:
            steps.append((None, [ready[0]]))              # compute-only step (L230)
            c_done.add(ready[0])
            continue
        _, kind, idx, t_comm = min(cands)                 # highest profit, then kind, then index
        fill, total = [], 0.0
        for t in ready:
            if total >= gamma * t_comm:
                break
            fill.append(t)
            total += t_c
        steps.append(((kind, idx), fill))
        c_done.update(fill)
        if kind == AG_KV:
            kv_done.add(idx)
            kv_next += 1
        elif kind == AG_Q:
            q_done.add(idx)
            q_next += 1
        else:
            rs_done.add(idx)
    return steps


def compute_order(steps):
    """The sequence of compute tasks (i, j) a step list executes."""
    return [t for _, fill in steps for t in fill]


def tile_list(n, a, b, kvr, g, order_ij):
    """Execution-ordered tiles (u, v, i, j) of GPU g: for each compute task C-i-j in schedule
    order, every (Q_u chunk i, KV_v chunk j) of the tile, u-major."""
    r, c = g // a, g % a
    IQ = list(range(r * a, (r + 1) * a))
    IKV = [c + t * a for t in range(b)] if kvr else list(range(c * b, (c + 1) * b))
    return [(u, v, i, j) for (i, j) in order_ij for u in IQ for v in IKV]
