"""The CPU oracle under AddressSanitizer + UndefinedBehaviorSanitizer: oracle/sanitize_driver.c
includes oracle/vmat_oracle.c, calls every entry point on a small seeded problem and must exit 0 with a clean stderr."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_runs_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "sanitize_driver")
    subprocess.run(["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                    "-fno-omit-frame-pointer", "-ffp-contract=off", os.path.join(ROOT, "oracle", "sanitize_driver.c"),
                    "-o", exe, "-lm"], check=True)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    res = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    assert "sanitize_driver ok" in res.stdout
    assert "ERROR" not in res.stderr and "runtime error" not in res.stderr, res.stderr[-2000:]
