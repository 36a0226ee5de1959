"""Thin ctypes binding of libmesh_attn.so (include/mesh_attn.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  There is no fallback: if the
shared library is missing this module raises at import, and compute calls on a machine
without a CUDA device raise MeshAttnError(ECUDA).
PyTorch appears only as the owner of device memory and streams (``tensor.data_ptr()``,
``torch.cuda.current_stream()``).
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_LIB_PATH = Path(__file__).resolve().parent / "libmesh_attn.so"
if not _LIB_PATH.exists():
    raise ImportError(
        f"{_LIB_PATH} is missing: build it with `python -m paper_2512_20968_b200.build` "
        "(or __graft_entry__.build()). There is no CPU or PyTorch fallback."
    )
lib = C.CDLL(str(_LIB_PATH))

OK, EINVAL, EUNSUPPORTED, EWORKSPACE, ECUDA, ENOMEM = 0, -1, -2, -3, -4, -5
(Q_PARTIAL_O_BYTES, Q_PARTIAL_LSE_BYTES, Q_SLOTS_PER_GPU, Q_FLOPS_FWD, Q_FLOPS_BWD, Q_WAVES, Q_MERGE_BYTES,
 Q_FWD_ITEMS_PER_GPU, Q_BWD_ITEMS_PER_GPU, Q_BLOCKS_FWD, Q_COMM_UNITS, Q_HAS_DEVICE, Q_BWD_WS_BYTES,
 Q_MESH_COMM_BYTES_FWD, Q_MESH_COMM_BYTES_BWD, Q_RING_COMM_BYTES_FWD, Q_USP_LANES, Q_USP_A2A_BYTES_FWD, Q_BWD_PAIRED, Q_GOO_PARTIAL_O_BYTES, Q_GOO_PARTIAL_LSE_BYTES, Q_GOO_COMM_BYTES, Q_FWD_PAIRED) = range(23)
TASK_AG_KV, TASK_AG_Q, TASK_RS_Q, TASK_C, TASK_RS_KV = range(5)


class PlanDesc(C.Structure):
    _fields_ = [
        ("n", C.c_int32), ("a", C.c_int32), ("b", C.c_int32),
        ("batch", C.c_int32), ("seq_total", C.c_int32), ("heads_q", C.c_int32), ("heads_kv", C.c_int32), ("head_dim", C.c_int32),
        ("causal", C.c_int32), ("kvr", C.c_int32), ("seq_layout", C.c_int32), ("order", C.c_int32),
        ("k_q", C.c_int32), ("k_kv", C.c_int32),
        ("gamma", C.c_float), ("t_ag_q", C.c_float), ("t_ag_kv", C.c_float), ("t_rs_q", C.c_float), ("t_c", C.c_float),
        ("softmax_scale", C.c_float),
        ("tensor_layout", C.c_int32), ("partial_mode", C.c_int32), ("precision", C.c_int32),
        ("usp_lanes", C.c_int32), ("bwd_pairing", C.c_int32), ("bwd_piece_blocks", C.c_int32), ("out_dtype", C.c_int32), ("fwd_pairing", C.c_int32),
    ]


class HostIO(C.Structure):
    _fields_ = [(name, C.c_void_p) for name in (
        "Q_host", "K_host", "V_host", "dO_host", "O_host", "lse_host", "dQ_host", "dK_host", "dV_host",
        "d_Q", "d_K", "d_V", "d_dO", "d_O", "d_lse", "d_bwd_ws", "d_dQ", "d_dK", "d_dV", "d_partial_O", "d_partial_lse")]


_P = C.c_void_p
_I32P = C.POINTER(C.c_int32)
lib.mesh_attn_plan_create.argtypes = [C.POINTER(PlanDesc), C.POINTER(_P)]
lib.mesh_attn_plan_destroy.argtypes = [_P]
lib.mesh_attn_plan_destroy.restype = None
lib.mesh_attn_plan_am.argtypes = [_P, _I32P]
lib.mesh_attn_plan_footprint.argtypes = [_P, C.c_int32, _I32P, _I32P]
lib.mesh_attn_plan_tiles.argtypes = [_P, C.c_int32, _I32P, C.c_int32, _I32P]
lib.mesh_attn_plan_steps.argtypes = [_P, C.c_int32, _I32P, C.c_int32, _I32P]
lib.mesh_attn_plan_query.argtypes = [_P, C.c_int32, C.POINTER(C.c_int64)]
lib.mesh_attn_plan_timeline.argtypes = [_P, C.c_int32] + [C.POINTER(C.c_double)] * 3
lib.mesh_attn_plan_tam_units.argtypes = [_P, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
lib.mesh_attn_tile_fwd.argtypes = [_P, C.c_int32, C.c_int32, _P, _P, _P, _P, _P, _P]
lib.mesh_attn_merge.argtypes = [_P, C.c_int32, _P, _P, _P, _P, _P]
lib.mesh_attn_bwd_preprocess.argtypes = [_P] * 6
lib.mesh_attn_tile_bwd.argtypes = [_P, C.c_int32, C.c_int32] + [_P] * 9
lib.mesh_attn_forward.argtypes = [_P] * 9
lib.mesh_attn_forward_goo.argtypes = [_P, C.c_int32] + [_P] * 8 + [C.c_int64, C.c_int32, C.c_int32, _P]
lib.mesh_attn_backward.argtypes = [_P] * 12
lib.mesh_attn_backward_goo.argtypes = [_P, C.c_int32] + [_P] * 9 + [C.c_int64, C.c_int32, C.c_int32, _P]
lib.mesh_attn_rank_fwd.argtypes = [_P, C.c_int32] + [_P] * 6
lib.mesh_attn_rank_merge.argtypes = [_P] * 6
lib.mesh_attn_rank_merge_peers.argtypes = [_P, C.POINTER(_P), C.POINTER(_P), _P, _P, _P]
lib.mesh_attn_rank_bwd_preprocess.argtypes = [_P] * 6
lib.mesh_attn_rank_sum_peers.argtypes = [_P, C.POINTER(_P), C.c_int32, C.c_int64, _P, _P]
lib.mesh_attn_rank_bwd.argtypes = [_P, C.c_int32] + [_P] * 9
lib.mesh_attn_step_host.argtypes = [_P, C.POINTER(HostIO), _P]
lib.mesh_attn_plan_health.argtypes = [_P]
lib.mesh_attn_forward_static.argtypes = [_P] * 7
lib.mesh_attn_forward_static_limits.argtypes = [_P, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
lib.mesh_attn_forward_static_poison.argtypes = [_P, C.c_uint32, _P]
lib.mesh_attn_launch_count.restype = C.c_int64
lib.mesh_attn_profile_enable.argtypes = [C.c_int32, C.c_int32]
lib.mesh_attn_profile_read.argtypes = [C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
lib.mesh_attn_strerror.restype = C.c_char_p
lib.mesh_attn_strerror.argtypes = [C.c_int]
lib.mesh_attn_last_error.restype = C.c_char_p

EXPORTED = [
    "mesh_attn_plan_create", "mesh_attn_plan_destroy", "mesh_attn_plan_am", "mesh_attn_plan_footprint", "mesh_attn_plan_tiles",
    "mesh_attn_plan_steps", "mesh_attn_plan_query", "mesh_attn_plan_tam_units", "mesh_attn_plan_timeline", "mesh_attn_tile_fwd", "mesh_attn_merge", "mesh_attn_bwd_preprocess",
    "mesh_attn_tile_bwd", "mesh_attn_forward", "mesh_attn_forward_goo", "mesh_attn_backward_goo", "mesh_attn_backward", "mesh_attn_step_host", "mesh_attn_launch_count", "mesh_attn_plan_health",
    "mesh_attn_profile_enable", "mesh_attn_profile_read", "mesh_attn_strerror", "mesh_attn_last_error",
    "mesh_attn_rank_fwd", "mesh_attn_rank_merge", "mesh_attn_rank_merge_peers", "mesh_attn_rank_sum_peers", "mesh_attn_rank_bwd_preprocess", "mesh_attn_rank_bwd",
    "mesh_attn_forward_static", "mesh_attn_forward_static_limits", "mesh_attn_forward_static_poison",
]
K_TILE_FWD, K_MERGE, K_BWD_PREPROCESS, K_TILE_BWD = range(4)


class MeshAttnError(RuntimeError):
    def __init__(self, status: int):
        self.status = status
        super().__init__(f"{lib.mesh_attn_strerror(status).decode()} ({status}): {lib.mesh_attn_last_error().decode()}")


def _check(status: int):
    if status != OK:
        raise MeshAttnError(status)


def _ptr(t):
    """device/host pointer of a torch tensor, numpy array, int or None"""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch

        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


class Plan:
    """mesh_attn_plan: host planner + device work lists.  Keyword arguments are mesh_attn_plan_desc fields."""

    def __init__(self, **kw):
        d = PlanDesc()
        for k, v in kw.items():
            if not hasattr(d, k):
                raise TypeError(f"unknown plan field {k}")
            setattr(d, k, v)
        if not d.n:
            d.n = d.a * d.b
        self.desc = d
        self._h = _P()
        _check(lib.mesh_attn_plan_create(C.byref(d), C.byref(self._h)))

    def close(self):
        if getattr(self, "_h", None) and lib is not None:
            lib.mesh_attn_plan_destroy(self._h)
        self._h = None

    __del__ = close

    # ---- planner queries (host) ----
    def query(self, what: int) -> int:
        v = C.c_int64()
        _check(lib.mesh_attn_plan_query(self._h, what, C.byref(v)))
        return v.value

    def health(self):
        """raises MeshAttnError(ECUDA) if a kernel of this plan reported a fault (synchronise the stream first)"""
        _check(lib.mesh_attn_plan_health(self._h))

    def timeline(self, backward: bool = False):
        """(makespan, serial time, exposed communication) of the step list in the plan's cost units"""
        m, s, e = C.c_double(), C.c_double(), C.c_double()
        _check(lib.mesh_attn_plan_timeline(self._h, int(backward), C.byref(m), C.byref(s), C.byref(e)))
        return m.value, s.value, e.value

    def tam_units(self, gpus_per_node: int, alpha: int, node: int = 0):
        """(Q-dimension, KV-dimension) inter-node units of `node` under the alpha-wide node tile"""
        q, kv = C.c_int64(), C.c_int64()
        _check(lib.mesh_attn_plan_tam_units(self._h, gpus_per_node, alpha, node, C.byref(q), C.byref(kv)))
        return q.value, kv.value

    def am(self) -> np.ndarray:
        n = self.desc.n
        out = np.empty((n, n), dtype=np.int32)
        _check(lib.mesh_attn_plan_am(self._h, out.ctypes.data_as(_I32P)))
        return out

    def footprint(self, g: int):
        iq = np.empty(self.desc.a, dtype=np.int32)
        ikv = np.empty(self.desc.b, dtype=np.int32)
        _check(lib.mesh_attn_plan_footprint(self._h, g, iq.ctypes.data_as(_I32P), ikv.ctypes.data_as(_I32P)))
        return iq, ikv

    def tiles(self, g: int) -> np.ndarray:
        cnt = C.c_int32()
        st = lib.mesh_attn_plan_tiles(self._h, g, None, 0, C.byref(cnt))
        if st not in (OK, EWORKSPACE):
            _check(st)
        out = np.empty((cnt.value, 4), dtype=np.int32)
        _check(lib.mesh_attn_plan_tiles(self._h, g, out.ctypes.data_as(_I32P), cnt.value, C.byref(cnt)))
        return out

    def steps(self, backward: bool = False) -> np.ndarray:
        cnt = C.c_int32()
        st = lib.mesh_attn_plan_steps(self._h, int(backward), None, 0, C.byref(cnt))
        if st not in (OK, EWORKSPACE):
            _check(st)
        out = np.empty((cnt.value, 4), dtype=np.int32)
        _check(lib.mesh_attn_plan_steps(self._h, int(backward), out.ctypes.data_as(_I32P), cnt.value, C.byref(cnt)))
        return out

    # ---- hot path (device pointers) ----
    def tile_fwd(self, g_first, g_count, Q, K, V, partial_O, partial_lse, stream=None):
        _check(lib.mesh_attn_tile_fwd(self._h, g_first, g_count, _ptr(Q), _ptr(K), _ptr(V), _ptr(partial_O), _ptr(partial_lse), _stream(stream)))

    def merge(self, q_group, partial_O, partial_lse, O, lse, stream=None):
        _check(lib.mesh_attn_merge(self._h, q_group, _ptr(partial_O), _ptr(partial_lse), _ptr(O), _ptr(lse), _stream(stream)))

    def bwd_preprocess(self, O, dO, lse, bwd_ws, stream=None):
        _check(lib.mesh_attn_bwd_preprocess(self._h, _ptr(O), _ptr(dO), _ptr(lse), _ptr(bwd_ws), _stream(stream)))

    def tile_bwd(self, g_first, g_count, Q, K, V, dO, bwd_ws, dQ, dK, dV, stream=None):
        _check(lib.mesh_attn_tile_bwd(self._h, g_first, g_count, _ptr(Q), _ptr(K), _ptr(V), _ptr(dO), _ptr(bwd_ws),
                                      _ptr(dQ), _ptr(dK), _ptr(dV), _stream(stream)))

    def forward(self, Q, K, V, O, lse, partial_O, partial_lse, stream=None):
        _check(lib.mesh_attn_forward(self._h, _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(lse), _ptr(partial_O), _ptr(partial_lse), _stream(stream)))

    def forward_static(self, Q, K, V, O, lse, stream=None):
        """forward() with the partial (O, lse) scratch in the library's built-in device array: allocates nothing; plans beyond
        forward_static_limits()[1] bytes raise MeshAttnError(EUNSUPPORTED); calls that overlap on the GPU race on the array"""
        _check(lib.mesh_attn_forward_static(self._h, _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(lse), _stream(stream)))

    def forward_static_limits(self):
        """(scratch bytes a forward_static of this plan uses, bytes the built-in array holds)"""
        need, cap = C.c_int64(), C.c_int64()
        _check(lib.mesh_attn_forward_static_limits(self._h, C.byref(need), C.byref(cap)))
        return need.value, cap.value

    def forward_static_poison(self, word=0x7FC00000, stream=None):
        """test hook: fill the built-in scratch array with `word` (default: a NaN)"""
        _check(lib.mesh_attn_forward_static_poison(self._h, word, _stream(stream)))

    def forward_goo(self, q_group, Q, K, V, O, lse, partial_O, partial_lse, comm_ws=None, comm_repeat=0, overlap=True, stream=None):
        nbytes = 0 if comm_ws is None else comm_ws.numel() * comm_ws.element_size()
        _check(lib.mesh_attn_forward_goo(self._h, q_group, _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(lse), _ptr(partial_O), _ptr(partial_lse),
                                         _ptr(comm_ws), nbytes, comm_repeat, int(bool(overlap)), _stream(stream)))

    def backward_goo(self, q_group, Q, K, V, dO, bwd_ws, dQ, dK, dV, comm_ws=None, comm_repeat=0, overlap=True, stream=None):
        nbytes = 0 if comm_ws is None else comm_ws.numel() * comm_ws.element_size()
        _check(lib.mesh_attn_backward_goo(self._h, q_group, _ptr(Q), _ptr(K), _ptr(V), _ptr(dO), _ptr(bwd_ws), _ptr(dQ), _ptr(dK), _ptr(dV),
                                          _ptr(comm_ws), nbytes, comm_repeat, int(bool(overlap)), _stream(stream)))

    def backward(self, Q, K, V, O, dO, lse, bwd_ws, dQ, dK, dV, stream=None):
        _check(lib.mesh_attn_backward(self._h, _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(dO), _ptr(lse), _ptr(bwd_ws),
                                      _ptr(dQ), _ptr(dK), _ptr(dV), _stream(stream)))

    # ---- per-rank calls (one GPU of a real n-GPU job; tensors hold the rank's gathered partitions only) ----
    def rank_fwd(self, g, Q_loc, K_loc, V_loc, partial_O, partial_lse, stream=None):
        _check(lib.mesh_attn_rank_fwd(self._h, g, _ptr(Q_loc), _ptr(K_loc), _ptr(V_loc), _ptr(partial_O), _ptr(partial_lse), _stream(stream)))

    def rank_merge(self, partial_O_recv, partial_lse_recv, O_own, lse_own, stream=None):
        _check(lib.mesh_attn_rank_merge(self._h, _ptr(partial_O_recv), _ptr(partial_lse_recv), _ptr(O_own), _ptr(lse_own), _stream(stream)))

    def rank_merge_peers(self, peer_partial_O, peer_partial_lse, O_own, lse_own, stream=None):
        """peer_partial_O / peer_partial_lse: sequences of `a` tensors or device addresses (member k's partial for this rank's partition)"""
        m = len(peer_partial_O)
        po = (_P * m)(*[_ptr(t) for t in peer_partial_O])
        pl = (_P * m)(*[_ptr(t) for t in peer_partial_lse])
        _check(lib.mesh_attn_rank_merge_peers(self._h, po, pl, _ptr(O_own), _ptr(lse_own), _stream(stream)))

    def rank_sum_peers(self, peers, out, stream=None):
        """out = sum of the fp32 buffers `peers` (tensors with out's element count, or device addresses)"""
        tab = (_P * len(peers))(*[_ptr(t) for t in peers])
        _check(lib.mesh_attn_rank_sum_peers(self._h, tab, len(peers), out.numel(), _ptr(out), _stream(stream)))

    def rank_bwd_preprocess(self, O_own, dO_own, lse_own, ws_own, stream=None):
        _check(lib.mesh_attn_rank_bwd_preprocess(self._h, _ptr(O_own), _ptr(dO_own), _ptr(lse_own), _ptr(ws_own), _stream(stream)))

    def rank_bwd(self, g, Q_loc, K_loc, V_loc, dO_loc, ws_loc, dQ_loc, dK_loc, dV_loc, stream=None):
        _check(lib.mesh_attn_rank_bwd(self._h, g, _ptr(Q_loc), _ptr(K_loc), _ptr(V_loc), _ptr(dO_loc), _ptr(ws_loc),
                                      _ptr(dQ_loc), _ptr(dK_loc), _ptr(dV_loc), _stream(stream)))

    def step_host(self, stream=None, **buffers):
        io = HostIO()
        for k, v in buffers.items():
            if not hasattr(io, k):
                raise TypeError(f"unknown host-io field {k}")
            setattr(io, k, _ptr(v))
        _check(lib.mesh_attn_step_host(self._h, C.byref(io), _stream(stream)))


def profile_enable(on: bool, capacity: int = 4096):
    _check(lib.mesh_attn_profile_enable(int(on), capacity))


def profile_read(kind: int):
    """(total milliseconds, launches) of the recorded launches of `kind`; synchronise the stream first."""
    ms, cnt = C.c_double(), C.c_int64()
    _check(lib.mesh_attn_profile_read(kind, C.byref(ms), C.byref(cnt)))
    return ms.value, cnt.value


def launch_count() -> int:
    return int(lib.mesh_attn_launch_count())
