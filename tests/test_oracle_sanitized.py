"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: oracle/rpa_oracle.c is
rebuilt with -fsanitize=address,undefined into a temporary .so and every pin test of tests/test_oracle_pins*.py is run
against THAT build in a subprocess (libasan preloaded into the interpreter).  Any out-of-bounds access, use after free,
signed overflow or misaligned access in the checker aborts the subprocess."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

RUNNER = """
import sys
sys.path.insert(0, {root!r})
import oracle
oracle._build = lambda: {lib!r}      # oracle.lib() loads whatever _build() returns
assert oracle.lib()._name == {lib!r}
import pytest
sys.exit(pytest.main(["-q", "-x", "-p", "no:cacheprovider", "tests/test_oracle_pins.py", "tests/test_oracle_pins_optical.py",
                      "tests/test_oracle_pins_orbitals.py", "tests/test_oracle_pins_real_axis.py"]))
"""


def _gcc_file(name):
    try:
        p = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True, check=True).stdout.strip()
    except (OSError, subprocess.CalledProcessError):
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_pins_pass_under_asan_and_ubsan(tmp_path):
    asan = _gcc_file("libasan.so")
    if asan is None:
        pytest.skip("gcc / libasan not available")
    lib = str(tmp_path / "librpa_oracle_san.so")
    src = os.path.join(ROOT, "oracle", "rpa_oracle.c")
    cc = ["gcc", "-O1", "-g", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-fsanitize=address,undefined",
          "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-o", lib, src, "-lm"]
    r = subprocess.run(cc, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    env = dict(os.environ, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", OMP_NUM_THREADS="4")
    run = subprocess.run([sys.executable, "-c", RUNNER.format(root=ROOT, lib=lib)], cwd=ROOT, env=env, capture_output=True,
                         text=True, timeout=900)
    tail = run.stdout[-3000:] + run.stderr[-3000:]
    assert run.returncode == 0, tail
    assert "ERROR: AddressSanitizer" not in tail and "runtime error:" not in tail, tail
    assert " passed" in run.stdout
