"""the C oracle (and the CPU context baseline beside it) under AddressSanitizer and
UndefinedBehaviorSanitizer.  tests/c/oracle_sanitize_main.c drives every entry point on ragged random sets;
any sanitizer report aborts it (-fno-sanitize-recover)."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_sanitize")
    cmd = ["gcc", "-O1", "-g", "-std=gnu99", "-Wall", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-pthread",
           os.path.join(ROOT, "tests", "c", "oracle_sanitize_main.c"), os.path.join(ROOT, "oracle", "lcs_oracle.c"),
           os.path.join(ROOT, "oracle", "bitpar_cpu.c"), "-o", exe, "-lm"]
    b = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert b.returncode == 0, b.stderr[-3000:]
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, (r.stdout[-1000:], r.stderr[-3000:])
    assert "sanitized ok" in r.stdout
