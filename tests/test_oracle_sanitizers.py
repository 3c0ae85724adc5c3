"""SURVEY.md section 5 (sanitizer runs): the oracle and the host-side schedule builder of the Cholesky task graph under
AddressSanitizer + UndefinedBehaviorSanitizer (g++ -fsanitize=address,undefined -fno-sanitize-recover=all), each as one
translation unit with a small driver (tests/sanitize/).  compute-sanitizer for the device code is closed on the GPU pool
(DESIGN.md section 11); this covers what runs on the host."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
FLAGS = ["-O1", "-g", "-std=c++17", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"]


def _build_and_run(tmp_path, src, extra):
    gxx = shutil.which("g++")
    if gxx is None:
        pytest.skip("g++ not available")
    exe = str(tmp_path / "a.out")
    r = subprocess.run([gxx] + FLAGS + extra + ["-o", exe, os.path.join(HERE, "sanitize", src), "-lm"], capture_output=True, text=True)
    if r.returncode != 0 and ("asan" in r.stderr or "ubsan" in r.stderr):
        pytest.skip("sanitizer runtime libraries not installed: " + r.stderr[-200:])
    assert r.returncode == 0, r.stderr[-2000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="4")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.stdout[-500:], r.stderr[-3000:])
    assert r.stdout.startswith("ok") and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
    return r.stdout


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    _build_and_run(tmp_path, "oracle_sanitize_main.cpp", ["-fopenmp"])


def test_schedule_builder_is_clean_under_asan_and_ubsan(tmp_path):
    cuda_inc = "/usr/local/cuda/include"
    if not os.path.exists(os.path.join(cuda_inc, "cuda_runtime.h")):
        pytest.skip("CUDA headers not found")
    out = _build_and_run(tmp_path, "schedule_sanitize_main.cpp", ["-x", "c++", "-I" + cuda_inc])
    assert int(out.split()[1]) > 10000
