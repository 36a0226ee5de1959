"""B200-native per-GPU compute core of Mesh-Attention (arxiv 2512.20968).

    from paper_2512_20968_b200 import Plan, plan_for, workloads

`Plan` wraps the C-ABI library (include/mesh_attn.h); everything on the hot path runs in
hand-written sm_100a CUDA kernels.  There is no CPU / PyTorch fallback.
"""
from . import workloads  # noqa: F401  (pure input generation, importable without the CUDA library)

_LAZY = ("Plan", "MeshAttnError", "launch_count", "binding")


def __getattr__(name):
    import importlib

    if name in _LAZY:
        binding = importlib.import_module(__name__ + ".binding")
        return binding if name == "binding" else getattr(binding, name)
    if name in ("plan_for", "Buffers", "runtime"):
        runtime = importlib.import_module(__name__ + ".runtime")
        return runtime if name == "runtime" else getattr(runtime, name)
    raise AttributeError(name)
