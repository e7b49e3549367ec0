"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer ("Race detection / sanitizers":
"oracle built with -fsanitize=address,undefined in tests").

oracle/pd_oracle.c is compiled a second time with -fsanitize=address,undefined -fno-sanitize-recover=all into pytest's
temporary directory, and the oracle's own pins (the tests/test_oracle_*.py files: every oracle function, every card key,
the worked events) are run once more in a child interpreter that loads that build (PD_ORACLE_LIB, with the sanitizer
run-times pre-loaded).  A heap overrun, a use after free, a signed overflow, a shift out of range, a misaligned or null
access anywhere in the checker ends the child with the sanitizer's report.  (The slowest statistical pin, 30 s without a
sanitizer, is left to the plain run.)"""
import glob
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _runtime(name):
    path = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return path if os.path.isabs(path) and os.path.exists(path) else None


def test_oracle_pins_under_asan_and_ubsan(tmp_path):
    if os.environ.get("PD_ORACLE_LIB"):
        pytest.skip("already inside the sanitizer run")
    asan, ubsan = _runtime("libasan.so"), _runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("gcc has no sanitizer run-times here")
    lib = str(tmp_path / "libpd_oracle_san.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-ffp-contract=off", "-std=c99", "-Wall", "-Wextra", "-shared", "-fPIC",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-o", lib,
                           os.path.join(ROOT, "oracle", "pd_oracle.c"), "-lm"])
    env = dict(os.environ, PD_ORACLE_LIB=lib, LD_PRELOAD=asan + ":" + ubsan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    # the child really runs on the sanitised build: it is the only library of the oracle it opens
    probe = "from oracle import pdo; pdo.lib(); print(open('/proc/self/maps').read())"
    maps = subprocess.run([sys.executable, "-c", probe], cwd=ROOT, env=env, capture_output=True, text=True, check=True).stdout
    assert "libpd_oracle_san.so" in maps and "libasan" in maps and "libubsan" in maps and "oracle/libpd_oracle.so" not in maps
    files = sorted(glob.glob(os.path.join(ROOT, "tests", "test_oracle_*.py")))
    files = [f for f in files if not f.endswith("test_oracle_sanitizers.py")]
    assert len(files) >= 10
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider",
                        "-k", "not poisson_is_the_quantile", *files], cwd=ROOT, env=env, capture_output=True, text=True)
    tail = (r.stdout[-3000:] + "\n" + r.stderr[-3000:])
    assert r.returncode == 0, tail
    assert " passed" in r.stdout and "failed" not in r.stdout, tail
    assert "AddressSanitizer" not in tail and "runtime error" not in tail, tail
