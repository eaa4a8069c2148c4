"""the oracle under AddressSanitizer + UndefinedBehaviorSanitizer.  tests/c/oracle_sanitize.c drives
every entry point of oracle/*.c on small inputs (frames, background rows, both light types, emitter normals, sub-ranges of
a frame, the per-pixel albedo plane, the encoder tail); any out-of-bounds access, use of uninitialised stack, signed
overflow or misaligned access aborts the run.  CPU only."""
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    exe = str(tmp_path / "oracle_sanitize")
    srcs = [os.path.join(ROOT, "oracle", f) for f in ("nbsdf_oracle.c", "nbsdf_oracle_paper.c", "nbsdf_oracle_encoder.c")]
    cmd = ["gcc", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
           "-ffp-contract=off", "-fopenmp", os.path.join(ROOT, "tests", "c", "oracle_sanitize.c")] + srcs + ["-o", exe, "-lm"]
    build = subprocess.run(cmd, capture_output=True, text=True)
    if build.returncode != 0 and "sanitize" in build.stderr and ("cannot find" in build.stderr or "unrecognized" in build.stderr):
        pytest.skip("this gcc has no sanitizer runtime: " + build.stderr.strip().splitlines()[-1])
    assert build.returncode == 0, build.stderr
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1", OMP_NUM_THREADS="2")
    p = subprocess.run([exe], capture_output=True, text=True, timeout=300, env=env)
    assert p.returncode == 0 and p.stdout.startswith("OK"), p.stdout + p.stderr
    assert "runtime error" not in p.stderr and "AddressSanitizer" not in p.stderr, p.stderr
