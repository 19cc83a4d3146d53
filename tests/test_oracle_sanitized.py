"""The oracle's pin suite once more with oracle.c built under AddressSanitizer + UndefinedBehaviorSanitizer
(-fsanitize=address,undefined -fno-sanitize-recover=all): an out-of-bounds row access, a use of an uninitialised
coefficient slot or signed overflow in an index would abort the child process.  SURVEY.md section 5."""
import glob
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _libasan():
    try:
        p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True, check=True).stdout.strip()
    except Exception:
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_pins_under_asan_ubsan():
    asan = _libasan()
    if asan is None:
        pytest.skip("gcc's libasan.so not found")
    env = dict(os.environ, ORACLE_SANITIZE="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4")
    tests = sorted(glob.glob(os.path.join(ROOT, "tests", "test_oracle_*.py")))
    tests = [t for t in tests if not t.endswith("test_oracle_sanitized.py")]
    assert len(tests) >= 5
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"] + tests,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0, (r.stdout[-3000:], r.stderr[-3000:])
    assert "passed" in r.stdout
    # the child really loaded the sanitized build
    assert os.path.exists(os.path.join(ROOT, "oracle", "liboracle_san.so"))
