"""The oracle's pins once more, against a build of oracle/su3_oracle.c with -fsanitize=address,undefined
(SURVEY.md section 5): an index map that reads or writes outside its arrays, a signed overflow in the site arithmetic
or a misaligned access would pass a value comparison by luck; under the sanitizers it aborts the child process.
The pins themselves are tests/test_oracle_pins.py, run unchanged in a child python with libasan preloaded."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _libasan():
    try:
        p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True, timeout=30).stdout.strip()
    except (OSError, subprocess.SubprocessError):
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_pins_under_asan_and_ubsan():
    asan = _libasan()
    if asan is None:
        pytest.skip("gcc has no libasan.so on this box")
    env = dict(os.environ, SU3_ORACLE_SANITIZED="1", LD_PRELOAD=asan, OMP_NUM_THREADS="4",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                        "-p", "no:cacheprovider"], capture_output=True, text=True, env=env, cwd=ROOT, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "failed" not in r.stdout, tail
    assert "AddressSanitizer" not in tail and "runtime error" not in tail, tail
    # the child really loaded the sanitized build
    chk = subprocess.run([sys.executable, "-c", "import oracle, ctypes; oracle.mul3; from oracle import su3_oracle as o; "
                          "o._load(); print(open('/proc/self/maps').read().count('libsu3oracle_san.so') > 0)"],
                         capture_output=True, text=True, env=env, cwd=ROOT, timeout=300)
    assert chk.stdout.strip().endswith("True"), chk.stdout + chk.stderr
