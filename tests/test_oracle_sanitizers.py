"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer (sanitizers): a copy of
oracle/ is built with -fsanitize=address,undefined and the operator pins are run against it in a subprocess with the
sanitizer runtimes preloaded.  Any out-of-bounds access, use of uninitialised stack memory caught by ASan, signed
overflow or misaligned access in oracle/tsm_oracle.c aborts that subprocess (halt_on_error) and fails this test.
(compute-sanitizer, the CUDA counterpart, is closed on the GPU pool: DESIGN.md section 8.)"""
import os
import shutil
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _runtime(name):
    try:
        p = subprocess.check_output(["gcc", f"-print-file-name={name}"], text=True).strip()
    except (OSError, subprocess.CalledProcessError):
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc sanitizer runtimes not installed")
    work = tmp_path / "san"
    work.mkdir()
    for d in ("oracle", "tests", "paper_1211_0126_b200"):
        shutil.copytree(os.path.join(ROOT, d), work / d,
                        ignore=shutil.ignore_patterns("*.so", "*.o", "build", "__pycache__", "csrc"))
    lib = work / "oracle" / "libtsm_oracle.so"
    subprocess.check_call(["gcc", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fopenmp", "-std=c11",
                           "-shared", "-fPIC", "-o", str(lib), str(work / "oracle" / "tsm_oracle.c"), "-lm"])
    os.utime(lib)   # newer than the source: oracle.build() keeps it
    env = dict(os.environ, LD_PRELOAD=f"{asan} {ubsan}", ASAN_OPTIONS="detect_leaks=0:halt_on_error=1",
               UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1", PYTHONPATH=str(work))
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_oracle_operator.py", "-x", "-q", "-p", "no:cacheprovider"],
                       cwd=str(work), env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-2000:])
    assert "passed" in r.stdout and "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr
