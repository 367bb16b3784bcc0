"""AddressSanitizer + UndefinedBehaviorSanitizer over the host code of the library (csrc/host_setup.cpp) and over the CPU
oracle: each is compiled together with a small driver (tests/sanitize_*_main.*) with
-fsanitize=address,undefined -fno-sanitize-recover and run; any report aborts with a non-zero exit code.
(compute-sanitizer runs of the device code are recorded in profiles/r02_sanitizers.md.)"""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]
ENV = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="2")


def _run(cmd, exe, tmp_path):
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr[-4000:]
    r = subprocess.run([exe], capture_output=True, text=True, env=ENV, cwd=tmp_path)
    assert r.returncode == 0 and "OK" in r.stdout and "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, \
        (r.stdout[-2000:], r.stderr[-4000:])
    return r.stdout


@pytest.mark.skipif(shutil.which("g++") is None, reason="g++ not available")
def test_host_setup_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "san_host")
    out = _run(["g++", "-std=c++17"] + SAN + [os.path.join(ROOT, "tests", "sanitize_host_main.cpp"),
                os.path.join(ROOT, "paper_2512_18010_b200", "csrc", "host_setup.cpp"), "-o", exe], exe, tmp_path)
    assert "nbf" in out


@pytest.mark.skipif(shutil.which("gcc") is None, reason="gcc not available")
def test_oracle_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "san_oracle")
    out = _run(["gcc", "-std=gnu99", "-fopenmp"] + SAN + [os.path.join(ROOT, "tests", "sanitize_oracle_main.c"),
                os.path.join(ROOT, "oracle", "scarf_oracle.c"), os.path.join(ROOT, "oracle", "angular_oracle.c"), "-lm", "-o", exe],
               exe, tmp_path)
    assert "path 0 vs path 1" in out
