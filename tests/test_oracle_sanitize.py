"""The oracle's C source under AddressSanitizer and UndefinedBehaviorSanitizer: every entry point on small
ragged grids, built and run as a stand-alone program (oracle/sanitize_main.c).  Values are pinned elsewhere; this looks for
out-of-bounds indices and undefined arithmetic in the code the parity tests trust."""
import os
import shutil
import subprocess

import pytest

ORACLE = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "oracle")


@pytest.mark.skipif(shutil.which("gcc") is None, reason="needs gcc")
def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "sanitize_main")
    build = subprocess.run(["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                            "-fno-omit-frame-pointer", "-Wall", "-o", exe, os.path.join(ORACLE, "sanitize_main.c"), "-lm"],
                           capture_output=True, text=True, cwd=ORACLE)
    assert build.returncode == 0, build.stderr[-3000:]
    run = subprocess.run([exe], capture_output=True, text=True, timeout=600,
                         env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1"))
    assert run.returncode == 0, (run.stdout[-1000:], run.stderr[-3000:])
    assert "checksum" in run.stdout and "runtime error" not in run.stderr and "AddressSanitizer" not in run.stderr
    assert "nan" not in run.stdout.lower() and "inf" not in run.stdout.lower()
