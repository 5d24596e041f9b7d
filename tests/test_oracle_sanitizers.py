"""The C oracle under AddressSanitizer + UndefinedBehaviorSanitizer (every parity claim stands on
oracle/mesh_ft_oracle.c, so it must not read out of bounds or rely on undefined behaviour).  tests/host/oracle_sanitize_main.c
includes the oracle's source, runs one forward and one backward per mode over frequencies that reach every branch, and
aborts on any sanitizer finding; its F(0) lines are also checked against the box's volume and area."""
import os
import shutil
import subprocess

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_forward_and_backward_are_clean_under_asan_and_ubsan(tmp_path):
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    exe = tmp_path / "oracle_sanitize"
    cmd = ["gcc", "-std=c11", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-Wall", "-Wextra",
           "-o", str(exe), os.path.join(HERE, "host", "oracle_sanitize_main.c"), "-lm"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0 and ("libasan" in r.stderr or "libubsan" in r.stderr or "cannot find -l" in r.stderr):
        pytest.skip("the sanitizer runtimes are not installed: " + r.stderr.strip().splitlines()[-1])
    assert r.returncode == 0, r.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    env.pop("LD_PRELOAD", None)
    run = subprocess.run([str(exe)], capture_output=True, text=True, env=env, timeout=120)
    assert run.returncode == 0, run.stdout + run.stderr
    assert "runtime error" not in run.stderr and "AddressSanitizer" not in run.stderr, run.stderr
    lines = run.stdout.strip().splitlines()
    assert abs(float(lines[0].split("=")[1]) - 0.7 * 0.45 * 0.3) < 1e-14                                 # F(0) = volume
    assert abs(float(lines[1].split("=")[1]) - 2 * (0.7 * 0.45 + 0.45 * 0.3 + 0.7 * 0.3)) < 1e-13        # F(0) = area
    assert lines[2].startswith("checksum ") and float(lines[2].split()[1]) == float(lines[2].split()[1])  # finite
