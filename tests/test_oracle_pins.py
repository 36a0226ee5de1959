"""Pins for the fp64 oracle (CPU only).  Each test ties oracle/ to something other than
itself: brute force on tiny inputs, closed forms, invariants fixed by the mathematics,
"any tiling merges to full attention", finite differences, and a
library second opinion (torch CPU fp64 softmax + autograd).

A plausible mistake anywhere in the oracle (dropped scale, wrong sign in dS, transposed
operand, wrong GQA head map, off-by-one in the causal rule) fails at least one of these.
"""
import math

import numpy as np
import pytest
import torch

from tests.util import bf16_bits, bits_to_f64

RNG = np.random.default_rng(20968)


def rand_bits(shape, scale=1.0):
    return bf16_bits(RNG.standard_normal(shape) * scale)


# ---------------------------------------------------------------------------
# brute force: softmax written as a ratio of plain sums (no max subtraction, no
# LSE), pure Python floats, tiny sizes.
# ---------------------------------------------------------------------------
def brute_fwd(q, k, v, scale, causal, pos, s, h, g):
    N, _, D = q.shape
    hk = h // g
    num = [0.0] * D
    den = 0.0
    for t in range(N):
        if causal and pos[t] > pos[s]:
            continue
        sc = 0.0
        for d in range(D):
            sc += float(q[s, h, d]) * float(k[t, hk, d])
        e = math.exp(scale * sc)
        den += e
        for d in range(D):
            num[d] += e * float(v[t, hk, d])
    if den == 0.0:
        return [0.0] * D, -math.inf
    return [x / den for x in num], math.log(den)


@pytest.mark.parametrize("causal,layout", [(False, "contiguous"), (True, "contiguous"), (True, "striped")])
def test_brute_force_tiny(oracle, causal, layout):
    n, L, Hq, Hkv, D = 4, 4, 4, 2, 8
    N = n * L
    q, k, v = rand_bits((N, Hq, D)), rand_bits((N, Hkv, D)), rand_bits((N, Hkv, D))
    pos = oracle.positions(n, L, layout)
    scale = 0.37
    rows = np.repeat(np.arange(N), Hq)
    heads = np.tile(np.arange(Hq), N)
    O, lse = oracle.fwd_rows(q, k, v, scale, causal, pos, rows, heads)
    qf, kf, vf = bits_to_f64(q), bits_to_f64(k), bits_to_f64(v)
    for i, (s, h) in enumerate(zip(rows, heads)):
        o_ref, lse_ref = brute_fwd(qf, kf, vf, scale, causal, pos, s, h, Hq // Hkv)
        assert np.allclose(O[i], o_ref, rtol=0, atol=1e-13)
        assert abs(lse[i] - lse_ref) < 1e-13


def test_positions_are_permutations_and_striped_rule(oracle):
    # striped = token positions interleaved across partitions.
    for n, L in [(4, 4), (9, 5), (16, 3)]:
        pc = oracle.positions(n, L, "contiguous")
        ps = oracle.positions(n, L, "striped")
        assert sorted(pc) == list(range(n * L)) and sorted(ps) == list(range(n * L))
        assert np.array_equal(pc, np.arange(n * L))
        # partition p holds positions {p, p+n, p+2n, ...}
        for p in range(n):
            assert list(ps[p * L:(p + 1) * L]) == [p + n * s for s in range(L)]


# ---------------------------------------------------------------------------
# closed forms
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("causal", [False, True])
def test_uniform_keys_give_mean_of_v(oracle, causal):
    n, L, H, D = 3, 8, 2, 16
    N = n * L
    q = rand_bits((N, H, D))
    k0 = rand_bits((1, H, D))
    k = np.repeat(k0, N, axis=0)
    v = rand_bits((N, H, D))
    pos = oracle.positions(n, L, "striped")
    scale = 0.25
    rows = np.repeat(np.arange(N), H)
    heads = np.tile(np.arange(H), N)
    O, lse = oracle.fwd_rows(q, k, v, scale, causal, pos, rows, heads)
    qf, kf, vf = bits_to_f64(q), bits_to_f64(k0), bits_to_f64(v)
    for i, (s, h) in enumerate(zip(rows, heads)):
        vis = (pos <= pos[s]) if causal else np.ones(N, bool)
        assert np.allclose(O[i], vf[vis, h].mean(axis=0), atol=1e-13)
        assert abs(lse[i] - (scale * qf[s, h] @ kf[0, h] + math.log(vis.sum()))) < 1e-12


def test_zero_query_gives_log_count(oracle):
    n, L, H, D = 2, 6, 1, 8
    N = n * L
    q = np.zeros((N, H, D), np.uint16)
    k, v = rand_bits((N, H, D)), rand_bits((N, H, D))
    pos = oracle.positions(n, L, "striped")
    _, lse = oracle.fwd_rows(q, k, v, 1.0, True, pos, np.arange(N), np.zeros(N, np.int32))
    assert np.allclose(lse, np.log(pos + 1.0), atol=1e-14)
    _, lse = oracle.fwd_rows(q, k, v, 1.0, False, pos, np.arange(N), np.zeros(N, np.int32))
    assert np.allclose(lse, math.log(N), atol=1e-14)


def test_dominant_key_selects_one_v_row(oracle):
    N, H, D = 32, 1, 8
    q = bf16_bits(np.ones((N, H, D)))
    kf = RNG.uniform(-0.5, 0.5, (N, H, D))
    t_star = 11
    kf[t_star] = 16.0            # score 128*scale vs |others| <= 4*scale
    k = bf16_bits(kf)
    v = rand_bits((N, H, D))
    scale = 0.5                  # gap >= 60 in the exponent
    O, lse = oracle.fwd_rows(q, k, v, scale, False, np.arange(N), np.arange(N), np.zeros(N, np.int32))
    assert np.allclose(O, bits_to_f64(v)[t_star, 0][None, :], atol=1e-15)
    assert np.allclose(lse, scale * 8 * 16.0, atol=1e-12)


def test_key_shift_invariance(oracle):
    # adding a vector u to every key leaves O unchanged and shifts LSE by scale*q.u;
    # values chosen so that k + u is exact in bf16.
    N, H, D = 24, 2, 8
    k0 = RNG.integers(-8, 9, (N, H, D)) * 0.25
    u = RNG.integers(-2, 3, (1, H, D)) * 0.5
    q = rand_bits((N, H, D))
    v = rand_bits((N, H, D))
    pos = np.arange(N)
    rows, heads = np.repeat(np.arange(N), H), np.tile(np.arange(H), N)
    for causal in (False, True):
        O0, l0 = oracle.fwd_rows(q, bf16_bits(k0), v, 0.3, causal, pos, rows, heads)
        O1, l1 = oracle.fwd_rows(q, bf16_bits(k0 + u), v, 0.3, causal, pos, rows, heads)
        assert np.allclose(O0, O1, atol=1e-13)
        shift = 0.3 * np.einsum("nhd,hd->nh", bits_to_f64(q), u[0]).reshape(-1)
        assert np.allclose(l1 - l0, shift, atol=1e-12)


def test_row_score_constant_invariance(oracle):
    # adding a constant to every score of a row (q -> q, k -> k + c*e0 with q[:,0] = 1) leaves O unchanged
    N, H, D = 16, 1, 4
    qf = RNG.integers(-4, 5, (N, H, D)) * 0.5
    qf[..., 0] = 1.0
    kf = RNG.integers(-4, 5, (N, H, D)) * 0.5
    v = rand_bits((N, H, D))
    kf2 = kf.copy()
    kf2[..., 0] += 3.0
    a = oracle.fwd_rows(bf16_bits(qf), bf16_bits(kf), v, 1.0, False, np.arange(N), np.arange(N), np.zeros(N, np.int32))
    b = oracle.fwd_rows(bf16_bits(qf), bf16_bits(kf2), v, 1.0, False, np.arange(N), np.arange(N), np.zeros(N, np.int32))
    assert np.allclose(a[0], b[0], atol=1e-13) and np.allclose(b[1] - a[1], 3.0, atol=1e-12)


# ---------------------------------------------------------------------------
# merge: identities and "any tiling of the assignment matrix merges to full attention"
# ---------------------------------------------------------------------------
def test_merge_identities(oracle):
    D = 8
    O1, O2 = RNG.standard_normal(D), RNG.standard_normal(D)
    # -inf partial is the identity
    O, lse = oracle.merge(np.stack([O1, np.zeros(D)]), [0.7, -np.inf])
    assert np.allclose(O, O1, atol=1e-15) and abs(lse - 0.7) < 1e-15
    # two identical partials: same O, lse + ln 2
    O, lse = oracle.merge(np.stack([O1, O1]), [0.7, 0.7])
    assert np.allclose(O, O1, atol=1e-15) and abs(lse - (0.7 + math.log(2))) < 1e-15
    # all -inf: (0, -inf), no NaN
    O, lse = oracle.merge(np.zeros((3, D)), [-np.inf] * 3)
    assert np.all(O == 0) and lse == -np.inf
    # weights are softmax of the lse's
    O, lse = oracle.merge(np.stack([O1, O2]), [1.0, 3.0])
    w = np.exp([1.0, 3.0]) / np.exp([1.0, 3.0]).sum()
    assert np.allclose(O, w[0] * O1 + w[1] * O2, atol=1e-15)
    assert abs(lse - math.log(math.exp(1.0) + math.exp(3.0))) < 1e-15
    # commutative / associative
    parts = RNG.standard_normal((5, D))
    lses = RNG.standard_normal(5) * 3
    Oa, la = oracle.merge(parts, lses)
    perm = RNG.permutation(5)
    Ob, lb = oracle.merge(parts[perm], lses[perm])
    O01, l01 = oracle.merge(parts[:2], lses[:2])
    Oc, lc = oracle.merge(np.concatenate([O01[None], parts[2:]]), np.concatenate([[l01], lses[2:]]))
    for Ox, lx in ((Ob, lb), (Oc, lc)):
        assert np.allclose(Oa, Ox, atol=1e-12) and abs(la - lx) < 1e-12


def _tilings(n, a, b):
    """key-partition subsets per simulated GPU column for the basic and KVR tilings, plus a random split."""
    basic = [list(range(c * b, (c + 1) * b)) for c in range(a)]
    kvr = [[c + t * a for t in range(b)] for c in range(a)]
    perm = list(RNG.permutation(n))
    cuts = sorted(RNG.choice(np.arange(1, n), size=2, replace=False))
    rnd = [perm[:cuts[0]], perm[cuts[0]:cuts[1]], perm[cuts[1]:]]
    per_pair = [[j] for j in range(n)]                                    # O_ij, lse_ij
    return {"basic": basic, "kvr": kvr, "random": rnd, "per_pair": per_pair}


@pytest.mark.parametrize("causal,layout", [(False, "contiguous"), (True, "contiguous"), (True, "striped")])
def test_any_tiling_merges_to_full(oracle, causal, layout):
    a, b, L, Hq, Hkv, D = 2, 3, 5, 2, 1, 8
    n = a * b
    N = n * L
    q, k, v = rand_bits((N, Hq, D)), rand_bits((N, Hkv, D)), rand_bits((N, Hkv, D))
    pos = oracle.positions(n, L, layout)
    rows, heads = np.repeat(np.arange(N), Hq), np.tile(np.arange(Hq), N)
    O_full, lse_full = oracle.fwd_rows(q, k, v, 0.35, causal, pos, rows, heads)
    part_of_row = np.arange(N) // L
    for name, subsets in _tilings(n, a, b).items():
        Os, ls = [], []
        for sub in subsets:
            sel = np.isin(part_of_row, sub).astype(np.uint8)
            O, l = oracle.fwd_rows(q, k, v, 0.35, causal, pos, rows, heads, key_sel=sel)
            Os.append(O)
            ls.append(l)
        Os, ls = np.stack(Os, 1), np.stack(ls, 1)          # [nq, m, D], [nq, m]
        for i in range(len(rows)):
            O, l = oracle.merge(Os[i], ls[i])
            assert np.allclose(O, O_full[i], atol=1e-12), name
            assert abs(l - lse_full[i]) < 1e-12, name


def test_striped_pair_with_no_visible_key(oracle):
    # striped pair (i, j) with j > i: local row s = 0 sees no key of partition j
    # (reading R5): partial = (0, -inf).
    n, L, D = 3, 4, 4
    N = n * L
    q, k, v = rand_bits((N, 1, D)), rand_bits((N, 1, D)), rand_bits((N, 1, D))
    pos = oracle.positions(n, L, "striped")
    sel = (np.arange(N) // L == 2).astype(np.uint8)      # keys of partition 2 only
    O, lse = oracle.fwd_rows(q, k, v, 1.0, True, pos, [0 * L + 0], [0], key_sel=sel)   # Q partition 0, s = 0
    assert lse[0] == -np.inf and np.all(O == 0)
    O, lse = oracle.fwd_rows(q, k, v, 1.0, True, pos, [0 * L + 1], [0], key_sel=sel)   # s = 1 sees key t = 0 only
    assert np.allclose(O[0], bits_to_f64(v)[2 * L + 0, 0], atol=1e-15)


# ---------------------------------------------------------------------------
# backward: finite differences of an independently written fp64 forward, library
# second opinion, closed form, global invariants
# ---------------------------------------------------------------------------
def np_forward(qf, kf, vf, scale, causal, pos, g):
    """independent fp64 forward on float arrays (einsum + masked softmax); returns O [N,Hq,D]."""
    N, Hq, D = qf.shape
    kk = np.repeat(kf, g, axis=1)
    vv = np.repeat(vf, g, axis=1)
    S = scale * np.einsum("shd,thd->hst", qf, kk)
    if causal:
        S = np.where(pos[None, None, :] <= pos[None, :, None], S, -np.inf)
    S = S - S.max(axis=-1, keepdims=True)
    P = np.exp(S)
    P /= P.sum(axis=-1, keepdims=True)
    return np.einsum("hst,thd->shd", P, vv)


@pytest.mark.parametrize("causal", [False, True])
def test_gradients_vs_finite_differences(oracle, causal):
    n, L, Hq, Hkv, D = 2, 4, 2, 1, 4
    N, g = n * L, Hq // Hkv
    q, k, v, do = rand_bits((N, Hq, D)), rand_bits((N, Hkv, D)), rand_bits((N, Hkv, D)), rand_bits((N, Hq, D))
    pos = oracle.positions(n, L, "striped")
    scale = 0.6
    qf, kf, vf, dof = (bits_to_f64(x) for x in (q, k, v, do))
    # the independent forward agrees with the oracle forward
    O_or, _ = oracle.fwd_full(q, k, v, scale, causal, pos)
    assert np.allclose(O_or, np_forward(qf, kf, vf, scale, causal, pos, g), atol=1e-12)

    def f(qa, ka, va):
        return float((np_forward(qa, ka, va, scale, causal, pos, g) * dof).sum())

    def fd(arr, which):
        out = np.zeros_like(arr)
        eps = 1e-6
        for idx in np.ndindex(arr.shape):
            ap, am = arr.copy(), arr.copy()
            ap[idx] += eps
            am[idx] -= eps
            args_p = {"q": (ap, kf, vf), "k": (qf, ap, vf), "v": (qf, kf, ap)}[which]
            args_m = {"q": (am, kf, vf), "k": (qf, am, vf), "v": (qf, kf, am)}[which]
            out[idx] = (f(*args_p) - f(*args_m)) / (2 * eps)
        return out

    rows, heads = np.repeat(np.arange(N), Hq), np.tile(np.arange(Hq), N)
    dq, _, _ = oracle.bwd_dq_rows(q, k, v, do, scale, causal, pos, rows, heads)
    assert np.allclose(dq.reshape(N, Hq, D), fd(qf, "q"), atol=1e-8)
    krows, kheads = np.repeat(np.arange(N), Hkv), np.tile(np.arange(Hkv), N)
    dk, dv = oracle.bwd_dkv_keys(q, k, v, do, scale, causal, pos, krows, kheads)
    assert np.allclose(dk.reshape(N, Hkv, D), fd(kf, "k"), atol=1e-8)
    assert np.allclose(dv.reshape(N, Hkv, D), fd(vf, "v"), atol=1e-8)


@pytest.mark.parametrize("causal,layout", [(False, "contiguous"), (True, "striped")])
def test_torch_fp64_second_opinion(oracle, causal, layout):
    n, L, Hq, Hkv, D = 4, 24, 4, 2, 16
    N, g = n * L, Hq // Hkv
    q, k, v, do = rand_bits((N, Hq, D)), rand_bits((N, Hkv, D)), rand_bits((N, Hkv, D)), rand_bits((N, Hq, D))
    pos = oracle.positions(n, L, layout)
    scale = D ** -0.5
    tq, tk, tv = (torch.tensor(bits_to_f64(x), requires_grad=True) for x in (q, k, v))
    tdo = torch.tensor(bits_to_f64(do))
    S = scale * torch.einsum("shd,thd->hst", tq, tk.repeat_interleave(g, dim=1))
    if causal:
        tp = torch.tensor(pos)
        S = S.masked_fill(tp[None, None, :] > tp[None, :, None], float("-inf"))
    O = torch.einsum("hst,thd->shd", torch.softmax(S, dim=-1), tv.repeat_interleave(g, dim=1))
    lse_t = torch.logsumexp(S, dim=-1)
    O.backward(tdo)
    O_or, lse_or = oracle.fwd_full(q, k, v, scale, causal, pos)
    assert np.allclose(O_or, O.detach().numpy(), atol=1e-12)
    assert np.allclose(lse_or, lse_t.detach().numpy(), atol=1e-12)
    rows, heads = np.repeat(np.arange(N), Hq), np.tile(np.arange(Hq), N)
    dq, lse2, _ = oracle.bwd_dq_rows(q, k, v, do, scale, causal, pos, rows, heads)
    assert np.allclose(dq.reshape(N, Hq, D), tq.grad.numpy(), atol=1e-11)
    assert np.allclose(lse2.reshape(N, Hq).T, lse_or, atol=1e-12)
    krows, kheads = np.repeat(np.arange(N), Hkv), np.tile(np.arange(Hkv), N)
    dk, dv = oracle.bwd_dkv_keys(q, k, v, do, scale, causal, pos, krows, kheads)
    assert np.allclose(dk.reshape(N, Hkv, D), tk.grad.numpy(), atol=1e-11)
    assert np.allclose(dv.reshape(N, Hkv, D), tv.grad.numpy(), atol=1e-11)
    # global invariants (rows of P sum to 1, rows of dS sum to 0), per KV head
    dof = bits_to_f64(do)
    for hk in range(Hkv):
        assert np.allclose(dv.reshape(N, Hkv, D)[:, hk].sum(0), dof[:, hk * g:(hk + 1) * g].sum((0, 1)), atol=1e-10)
        assert np.allclose(dk.reshape(N, Hkv, D)[:, hk].sum(0), 0.0, atol=1e-10)
    assert abs((bits_to_f64(q) * dq.reshape(N, Hq, D)).sum() - (bits_to_f64(k) * dk.reshape(N, Hkv, D)).sum()) < 1e-9


def test_sparse_do_probe_rows_subset(oracle):
    # dK/dV with dO non-zero on R rows only == sum restricted to those rows (linearity in dO)
    n, L, H, D = 2, 8, 1, 8
    N = n * L
    q, k, v = rand_bits((N, H, D)), rand_bits((N, H, D)), rand_bits((N, H, D))
    do = np.zeros((N, H, D), np.uint16)
    live = np.array([1, 6, 11])
    do[live] = rand_bits((3, H, D))
    pos = oracle.positions(n, L, "striped")
    kr, kh = np.arange(N), np.zeros(N, np.int32)
    full = oracle.bwd_dkv_keys(q, k, v, do, 0.4, True, pos, kr, kh)
    sub = oracle.bwd_dkv_keys(q, k, v, do, 0.4, True, pos, kr, kh, qs_rows=live)
    assert np.allclose(full[0], sub[0], atol=1e-14) and np.allclose(full[1], sub[1], atol=1e-14)


def test_uniform_keys_gradient_closed_form(oracle):
    # identical keys: P[s,t] = 1/#visible(s)  =>  dQ = 0, dV[t] = sum_{s sees t} dO[s]/#visible(s)
    n, L, H, D = 2, 5, 1, 8
    N = n * L
    q, v, do = rand_bits((N, H, D)), rand_bits((N, H, D)), rand_bits((N, H, D))
    k = np.repeat(rand_bits((1, H, D)), N, axis=0)
    pos = oracle.positions(n, L, "striped")
    dq, _, _ = oracle.bwd_dq_rows(q, k, v, do, 0.5, True, pos, np.arange(N), np.zeros(N, np.int32))
    assert np.allclose(dq, 0.0, atol=1e-13)
    _, dv = oracle.bwd_dkv_keys(q, k, v, do, 0.5, True, pos, np.arange(N), np.zeros(N, np.int32))
    dof = bits_to_f64(do)[:, 0]
    ref = np.zeros((N, D))
    for t in range(N):
        for s in range(N):
            if pos[t] <= pos[s]:
                ref[t] += dof[s] / (pos[s] + 1)
    assert np.allclose(dv, ref, atol=1e-13)
