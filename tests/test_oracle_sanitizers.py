"""The C oracle under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md section 5 "oracle under
-fsanitize=address,undefined"): a second build of oracle/rubix_oracle.c runs a cross-section of its own pins -- every
entry point is exercised (binning, sort, cells, spectra of every mode, cubes, convolutions, adjoints, noise) -- in a child
process started with libasan preloaded.  Any out-of-bounds access, signed overflow, misaligned access or invalid shift aborts
the child with a non-zero exit code."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FILES = ["tests/test_oracle_binning.py", "tests/test_oracle_spectrum.py", "tests/test_oracle_convolve.py",
         "tests/test_oracle_noise.py", "tests/test_oracle_obsgrid.py", "tests/test_oracle_varpsf.py"]
KEYWORDS = {"tests/test_oracle_gengrid.py": "prefix_integral or cube_is_the_sum or point_rule",
            "tests/test_oracle_fluxcons.py": "prefix or telescopes or cube_is_the_sum",
            "tests/test_oracle_adjoint.py": "dot_product or closed or linear"}


def _lib(name):
    path = subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True).stdout.strip()
    return path if os.path.isabs(path) and os.path.exists(path) else None


def test_oracle_pins_pass_under_asan_and_ubsan():
    asan = _lib("libasan.so")
    if asan is None:
        pytest.skip("gcc has no libasan on this machine")
    env = dict(os.environ, RUBIX_ORACLE_SANITIZE="1", LD_PRELOAD=asan, OMP_NUM_THREADS="4",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    base = [sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider"]
    r = subprocess.run(base + FILES, cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "passed" in r.stdout and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
    for f, k in KEYWORDS.items():
        r = subprocess.run(base + [f, "-k", k], cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
        assert r.returncode == 0, (f, r.stdout[-3000:] + r.stderr[-3000:])
        assert "passed" in r.stdout and "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
