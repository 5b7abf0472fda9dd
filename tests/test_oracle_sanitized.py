"""The oracle's C code under AddressSanitizer + UndefinedBehaviorSanitizer: the pin suite is run once
more in a subprocess against oracle/hardkv_oracle.c built with -fsanitize=address,undefined (libasan preloaded into the
interpreter).  A heap overflow, a use after free or undefined integer / shift behaviour anywhere on the paths the pins
drive aborts the subprocess."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib(name):
    out = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


def test_oracle_pins_under_asan_ubsan():
    asan, ubsan = _lib("libasan.so"), _lib("libubsan.so")
    if not asan:
        pytest.skip("gcc has no libasan on this box")
    env = dict(os.environ, HARDKV_ORACLE_SANITIZE="1", LD_PRELOAD=":".join(x for x in (asan, ubsan) if x),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               OMP_NUM_THREADS="2")
    # the pins that drive every oracle entry point: attention + merge (P1, P8), Top-p (P2-P5), rewrite / table / mask
    # (P9), retirement (P10, P11), temperature solve (P13), SNAPKV (P14), merging (P15), reuse steps (P16), query cache (P17)
    sel = "p1_ or p2_ or p3_ or p4_ or p5_ or p8_ or p9_ or p10_ or p13_identity or p14_ or p15_ or p16_ or p17_ or accum or empty_pool"
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                        "-k", sel, "-p", "no:cacheprovider"], cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert "passed" in r.stdout and "AddressSanitizer" not in tail and "runtime error" not in tail, tail
