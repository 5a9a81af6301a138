"""The oracles under AddressSanitizer + UndefinedBehaviorSanitizer -- -m "not gpu".

oracle/*.c are compiled together with tests/sanitize/driver.c (both precisions of real_t) with
`-fsanitize=address,undefined -fno-sanitize-recover=all` and run on small seeded inputs of every boundary mix; any
out-of-bounds access, use of freed memory, signed overflow or misaligned access aborts the run."""
import glob
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("defs", [[], ["-DORACLE_LONG_DOUBLE"]], ids=["double", "long_double"])
def test_oracles_under_asan_ubsan(tmp_path, defs):
    exe = str(tmp_path / "oracle_san")
    srcs = sorted(glob.glob(os.path.join(ROOT, "oracle", "*.c"))) + [os.path.join(ROOT, "tests", "sanitize", "driver.c")]
    cmd = ["gcc", "-std=c11", "-O1", "-g", "-ffp-contract=off", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-fno-omit-frame-pointer", *defs, *srcs, "-o", exe, "-lm"]
    subprocess.run(cmd, check=True)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert "sanitizer driver done, status 0" in r.stdout
