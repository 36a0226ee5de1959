"""Host sanitizer build: csrc/planner.cpp and oracle/mesh_attn_oracle.c compiled with
-fsanitize=address,undefined and driven by tests/sanitize/sanitize_main.cpp (BASELINE.json's five geometries and
structural variants through every planner call, refused descriptors, the oracle's four functions on a small problem).
compute-sanitizer is closed on the GPU pool, so the device code has no sanitizer run; this covers the host code."""
import os
import shutil
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
CSRC = ROOT / "paper_2512_20968_b200" / "csrc"


@pytest.mark.skipif(shutil.which("g++") is None or shutil.which("gcc") is None, reason="needs gcc / g++")
def test_planner_and_oracle_under_asan_ubsan(tmp_path):
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g", "-O1"]
    obj = tmp_path / "oracle.o"
    subprocess.check_call(["gcc", *san, "-std=c11", "-fopenmp", "-c", str(ROOT / "oracle" / "mesh_attn_oracle.c"), "-o", str(obj)])
    exe = tmp_path / "sanitize_main"
    subprocess.check_call(["g++", *san, "-std=c++17", f"-I{ROOT / 'include'}", f"-I{CSRC}", str(CSRC / "planner.cpp"),
                           str(ROOT / "tests" / "sanitize" / "sanitize_main.cpp"), str(obj), "-fopenmp", "-lm", "-o", str(exe)])
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0:halt_on_error=1", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "sanitize_main: ok" in r.stdout
    assert "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr and "LeakSanitizer" not in r.stderr, r.stderr[-4000:]
