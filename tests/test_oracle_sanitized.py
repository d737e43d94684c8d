"""The oracle pins once more against the oracle built with -fsanitize=address,undefined (SURVEY.md section 5:
"oracle built with -fsanitize=address,undefined").  CPU only.  A child pytest runs the test_oracle_*.py files
with ASR_ORACLE_SANITIZE=1 (oracle/__init__.py then builds and loads libasr_oracle_san.so) and libasan
preloaded; any heap overflow, use after free or undefined behaviour in asr_oracle.c aborts the child."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _runtime(name):
    try:
        p = subprocess.check_output(["gcc", "-print-file-name=" + name], text=True).strip()
    except Exception:
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


@pytest.mark.skipif(os.environ.get("ASR_ORACLE_SANITIZE") == "1", reason="already inside the sanitized child run")
def test_oracle_pins_hold_under_asan_ubsan():
    asan = _runtime("libasan.so")
    if asan is None:
        pytest.skip("gcc has no libasan on this machine")
    files = sorted(f for f in os.listdir(os.path.join(ROOT, "tests"))
                   if f.startswith("test_oracle_") and f.endswith(".py") and f != "test_oracle_sanitized.py")
    assert len(files) >= 5
    env = dict(os.environ, ASR_ORACLE_SANITIZE="1", LD_PRELOAD=asan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    cmd = [sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"] + \
          [os.path.join("tests", f) for f in files]
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "AddressSanitizer" not in tail and "runtime error" not in tail, tail
