"""The C oracle under AddressSanitizer + UndefinedBehaviorSanitizer: a small
driver (oracle/sanitize_driver.c) calls every entry point on deterministic inputs, edge cases
included; the sanitised binary must exit 0 with no report and print exactly what the plain build
prints (same flags otherwise, no FMA contraction)."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = [os.path.join(ROOT, "oracle", "oracle_fredec.c"), os.path.join(ROOT, "oracle", "sanitize_driver.c")]
CFLAGS = ["-O1", "-g", "-ffp-contract=off", "-Wall", "-Wextra", "-std=c11"]


def _build_and_run(tmp_path, name, extra):
    exe = str(tmp_path / name)
    subprocess.check_call(["gcc", *CFLAGS, *extra, *SRC, "-lm", "-o", exe])
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="halt_on_error=1")
    return subprocess.run([exe], capture_output=True, text=True, env=env, timeout=120)


def test_oracle_clean_under_asan_ubsan(tmp_path):
    plain = _build_and_run(tmp_path, "plain", [])
    san = _build_and_run(tmp_path, "san", ["-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                                           "-fno-omit-frame-pointer"])
    assert plain.returncode == 0, plain.stderr
    assert san.returncode == 0, san.stderr
    assert "ERROR" not in san.stderr and "runtime error" not in san.stderr, san.stderr
    assert san.stdout == plain.stdout
    lines = plain.stdout.strip().splitlines()
    assert lines[-1] == "rc=0" and any(l.startswith("trig 4") for l in lines)
    # the singular trial frequencies of the driver (f = 0 with a constant; f = a base frequency) give z = 0
    scan3 = [l for l in lines if l.startswith("scan d=4")][0].split()
    assert float(scan3[3]) == 0.0 and float(scan3[5]) == 0.0
    assert "edge found=1 idx0=40 idx1=-1" in plain.stdout
