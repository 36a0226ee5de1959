"""Build libmesh_attn.so (the C-ABI library) in-tree with nvcc for sm_100a.

    python -m paper_2512_20968_b200.build [--force]

nvcc cross-compiles without a GPU; the built .so is git-ignored but travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libmesh_attn.so"
OBJ = PKG / "build"
SOURCES = ["planner.cpp", "capi.cu", "tile_fwd.cu", "tile_bwd.cu", "aux_kernels.cu", "no_alloc.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v", f"-I{INCLUDE}", f"-I{CSRC}",
]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.sep not in c or os.path.exists(c)):
            return c
    raise RuntimeError("nvcc not found")


def _stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    deps = list(CSRC.glob("*")) + list(INCLUDE.glob("*.h")) + [Path(__file__)]
    return any(d.stat().st_mtime > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not _stale():
        return LIB
    OBJ.mkdir(exist_ok=True)
    nvcc = _nvcc()

    extra = os.environ.get("MESH_ATTN_NVCC_EXTRA", "").split()      # e.g. -DMESH_ATTN_POLY_OF_8=1 for tuning builds

    def compile_one(src: str):
        obj = OBJ / (src.rsplit(".", 1)[0] + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *extra, "-x", "cu", "-c", str(CSRC / src), "-o", str(obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        (OBJ / (src + ".log")).write_text(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed for {src}:\n{r.stdout}\n{r.stderr}")
        if verbose:
            print(r.stderr)
        return str(obj)

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    subprocess.check_call([nvcc, "-shared", "-o", str(tmp), *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    os.replace(tmp, LIB)
    return LIB


def kernel_source_hash(kernel: str) -> str:
    """sha256 (first 16 hex digits) of the sources that define `kernel` ("tile_fwd", "tile_bwd", "merge", ...): its .cu file and
    the shared headers.  profiles/*_traffic_*.md record it, so that bench.py can say whether a stored ncu capture still
    describes the kernel that runs."""
    import hashlib

    main = {"tile_fwd": "tile_fwd.cu", "tile_bwd": "tile_bwd.cu"}.get(kernel, "aux_kernels.cu")
    h = hashlib.sha256()
    for name in (main, "sm100.cuh", "tile_kernels.hpp", "plan.hpp"):
        h.update((CSRC / name).read_bytes())
    return h.hexdigest()[:16]


if __name__ == "__main__":
    if "--hash" in sys.argv:
        print(kernel_source_hash(sys.argv[sys.argv.index("--hash") + 1]))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
