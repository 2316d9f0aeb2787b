"""the oracle under AddressSanitizer + UndefinedBehaviorSanitizer.  The oracle is rebuilt with
-fsanitize=address,undefined and its pin tests (decode, attention, FP8 / retrieval, geometry, mask construction,
head schedule) run again in a child process that preloads libasan; any report fails the test.  (The CUDA side has no
such run: compute-sanitizer is closed on the GPU pool.)"""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PINS = ["tests/test_oracle_decode.py", "tests/test_oracle_attention.py", "tests/test_oracle_fp8_retrieve.py",
        "tests/test_oracle_geometry.py", "tests/test_oracle_mask_build.py", "tests/test_head_schedule.py"]


def test_oracle_pins_under_asan_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan is not installed")
    from oracle import build as obuild
    obuild.build(sanitize=True)
    env = dict(os.environ, CHORUS_ORACLE_SANITIZE="1", LD_PRELOAD=asan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=0:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4")
    out = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", *PINS], cwd=ROOT, env=env,
                         capture_output=True, text=True, timeout=1500)
    text = out.stdout + out.stderr
    assert "AddressSanitizer" not in text and "runtime error" not in text, text[-3000:]
    assert out.returncode == 0, text[-3000:]
    assert " passed" in out.stdout
