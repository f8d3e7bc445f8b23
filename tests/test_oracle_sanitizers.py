"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer, no GPU.

tests/helpers/oracle_sanitize_main.cpp calls every exported oracle function on small problems (both models, all
cost and noise kinds, ragged sizes, absent optional outputs); it is compiled together with the oracle source with
-fsanitize=address,undefined -fno-sanitize-recover=all, so an out-of-bounds access, a use after free, signed
overflow, a bad shift or cast, or a leak ends the run with a non-zero exit code."""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_sanitize")
    cmd = ["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-pthread", "-fsanitize=address,undefined",
           "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", f"-I{os.path.join(ROOT, 'oracle')}",
           os.path.join(ROOT, "tests", "helpers", "oracle_sanitize_main.cpp"),
           os.path.join(ROOT, "oracle", "ra_mppi_oracle.cpp"), "-o", exe]
    b = subprocess.run(cmd, capture_output=True, text=True)
    if b.returncode != 0 and "sanitize" in (b.stderr or "") and "cannot find" in b.stderr:
        pytest.skip("sanitizer runtime not installed")
    assert b.returncode == 0, b.stderr
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300,
                       env={**os.environ, "ASAN_OPTIONS": "detect_leaks=1:abort_on_error=0", "UBSAN_OPTIONS": "print_stacktrace=1"})
    assert r.returncode == 0, r.stdout + r.stderr
    assert "rc=0" in r.stdout and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
