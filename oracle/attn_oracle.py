"""fp64 CPU oracle for the Mesh-Attention compute core -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this module.  It never imports the product
package and shares no code with the CUDA path.

The arithmetic lives in ``mesh_attn_oracle.c`` (plain C, fp64, the definition of
softmax attention, and its derivative); this file is the ctypes
marshalling plus the two-line token-position map (DESIGN.md reading
R6) and thin loops that call the C rows functions.

Inputs are numpy ``uint16`` arrays holding bf16 bit patterns, layout ``[N, H, D]``
(one batch element), rows in partition-major order: row = p*L + s.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "mesh_attn_oracle.c"
_LIB = _HERE / "libmesh_attn_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", str(tmp), str(_SRC), "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        c = ctypes
        p = c.c_void_p
        lib.oracle_num_threads.restype = c.c_int
        lib.oracle_attn_fwd_rows.argtypes = [p, p, p, c.c_int64, c.c_int, c.c_int, c.c_int, c.c_double, c.c_int,
                                             p, p, c.c_int64, p, p, p, p]
        lib.oracle_attn_merge.argtypes = [c.c_int, c.c_int, p, p, p, p]
        lib.oracle_attn_bwd_dq_rows.argtypes = [p, p, p, p, c.c_int64, c.c_int, c.c_int, c.c_int, c.c_double, c.c_int,
                                                p, c.c_int64, p, p, p, p, p]
        lib.oracle_attn_bwd_dkv_keys.argtypes = [p, p, p, p, c.c_int64, c.c_int, c.c_int, c.c_int, c.c_double, c.c_int,
                                                 p, c.c_int64, p, p, p, c.c_int64, p, p, p, p]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _bits(x) -> np.ndarray:
    """Accept a numpy uint16 array (bf16 bits) or a torch CPU bf16 tensor."""
    if isinstance(x, np.ndarray):
        assert x.dtype == np.uint16
        return np.ascontiguousarray(x)
    import torch  # plumbing only: reinterpret bf16 bits

    assert x.dtype == torch.bfloat16 and x.device.type == "cpu"
    return np.ascontiguousarray(x.contiguous().view(torch.int16).numpy().view(np.uint16))


# --------------------------------------------------------------------------------------
# token positions (PAPER.md L278 striped layout "similar to Striped Attention";
# DESIGN.md reading R6).  Partition p holds local rows s = 0..L-1 at row p*L+s.
#   contiguous: pos = p*L + s           striped: pos = s*n + p
# --------------------------------------------------------------------------------------
def positions(n: int, L: int, seq_layout: str) -> np.ndarray:
    p, s = np.divmod(np.arange(n * L, dtype=np.int64), L)
    return p * L + s if seq_layout == "contiguous" else s * n + p


def fwd_rows(q, k, v, scale, causal, pos, qrows, qheads, key_sel=None):
    """O[nq, D] (fp64), LSE[nq] of the sampled (row, head) pairs, from the definition."""
    q, k, v = _bits(q), _bits(k), _bits(v)
    N, Hq, D = q.shape
    Hkv = k.shape[1]
    qrows = np.ascontiguousarray(qrows, dtype=np.int64)
    qheads = np.ascontiguousarray(qheads, dtype=np.int32)
    pos = np.ascontiguousarray(pos, dtype=np.int64)
    ks = None if key_sel is None else np.ascontiguousarray(key_sel, dtype=np.uint8)
    O = np.empty((len(qrows), D), dtype=np.float64)
    lse = np.empty(len(qrows), dtype=np.float64)
    _load().oracle_attn_fwd_rows(_ptr(q), _ptr(k), _ptr(v), N, Hq, Hkv, D, float(scale), int(causal),
                                 _ptr(pos), _ptr(ks), len(qrows), _ptr(qrows), _ptr(qheads), _ptr(O), _ptr(lse))
    return O, lse


def fwd_full(q, k, v, scale, causal, pos, heads=None):
    """O[N, len(heads), D], LSE[len(heads), N] for whole heads."""
    N, Hq, D = _bits(q).shape
    heads = list(range(Hq)) if heads is None else list(heads)
    rows = np.tile(np.arange(N, dtype=np.int64), len(heads))
    hh = np.repeat(np.asarray(heads, dtype=np.int32), N)
    O, lse = fwd_rows(q, k, v, scale, causal, pos, rows, hh)
    return O.reshape(len(heads), N, D).transpose(1, 0, 2).copy(), lse.reshape(len(heads), N)


def merge(O_parts, lse_parts):
    """Textbook LSE-weighted merge of m partials of one (row, head): ([m, D], [m]) -> ([D], scalar)."""
    O_parts = np.ascontiguousarray(O_parts, dtype=np.float64)
    lse_parts = np.ascontiguousarray(lse_parts, dtype=np.float64)
    m, D = O_parts.shape
    O = np.empty(D, dtype=np.float64)
    lse = np.empty(1, dtype=np.float64)
    _load().oracle_attn_merge(m, D, _ptr(O_parts), _ptr(lse_parts), _ptr(O), _ptr(lse))
    return O, float(lse[0])


def bwd_dq_rows(q, k, v, do, scale, causal, pos, qrows, qheads):
    """dQ[nq, D], LSE[nq], Delta[nq] of the sampled (row, head) pairs."""
    q, k, v, do = _bits(q), _bits(k), _bits(v), _bits(do)
    N, Hq, D = q.shape
    Hkv = k.shape[1]
    qrows = np.ascontiguousarray(qrows, dtype=np.int64)
    qheads = np.ascontiguousarray(qheads, dtype=np.int32)
    pos = np.ascontiguousarray(pos, dtype=np.int64)
    dq = np.empty((len(qrows), D), dtype=np.float64)
    lse = np.empty(len(qrows), dtype=np.float64)
    delta = np.empty(len(qrows), dtype=np.float64)
    _load().oracle_attn_bwd_dq_rows(_ptr(q), _ptr(k), _ptr(v), _ptr(do), N, Hq, Hkv, D, float(scale), int(causal),
                                    _ptr(pos), len(qrows), _ptr(qrows), _ptr(qheads), _ptr(dq), _ptr(lse), _ptr(delta))
    return dq, lse, delta


def bwd_dkv_keys(q, k, v, do, scale, causal, pos, krows, kheads, qs_rows=None):
    """dK[nk, D], dV[nk, D] of the sampled (key row, KV head) pairs.

    ``qs_rows``: the query rows summed over (default: all N; the rows with non-zero dO
    for the sparse-dO probe -- gradients are linear in dO, rows with dO = 0 add nothing).
    """
    qb, kb, vb, dob = _bits(q), _bits(k), _bits(v), _bits(do)
    N, Hq, D = qb.shape
    Hkv = kb.shape[1]
    g = Hq // Hkv
    krows = np.ascontiguousarray(krows, dtype=np.int64)
    kheads = np.ascontiguousarray(kheads, dtype=np.int32)
    pos = np.ascontiguousarray(pos, dtype=np.int64)
    qs = np.arange(N, dtype=np.int64) if qs_rows is None else np.ascontiguousarray(qs_rows, dtype=np.int64)
    # LSE and Delta of every (query head in the touched groups, summed-over row)
    lse_all = np.zeros((Hq, N), dtype=np.float64)
    delta_all = np.zeros((Hq, N), dtype=np.float64)
    for hk in sorted(set(int(x) for x in kheads)):
        for h in range(hk * g, (hk + 1) * g):
            _, lse, delta = bwd_dq_rows(qb, kb, vb, dob, scale, causal, pos, qs, np.full(len(qs), h, dtype=np.int32))
            lse_all[h, qs] = lse
            delta_all[h, qs] = delta
    dk = np.empty((len(krows), D), dtype=np.float64)
    dv = np.empty((len(krows), D), dtype=np.float64)
    _load().oracle_attn_bwd_dkv_keys(_ptr(qb), _ptr(kb), _ptr(vb), _ptr(dob), N, Hq, Hkv, D, float(scale), int(causal),
                                     _ptr(pos), len(qs), _ptr(qs), _ptr(lse_all), _ptr(delta_all),
                                     len(krows), _ptr(krows), _ptr(kheads), _ptr(dk), _ptr(dv))
    return dk, dv
