"""SURVEY.md sec. 8(f) NEXT-4, throughput half, as a MEASUREMENT: tests/cuda/tcgen05_kind_rate.cu issues
the decoder's own tcgen05.mma form (M = 128, A in TMEM, B in swizzled shared memory, fp32 accumulate) with kind::f16 and with
kind::f8f6f4 / e4m3 operands, checks the e4m3 products exactly, and times 4096 back-to-back instructions on every SM.
Four issue patterns: every instruction into the same accumulator tile (the K steps of one layer: a dependent chain), two
accumulator tiles alternating, the latter with the A operand in shared memory, and TWO issuing warps with a tile each.
Asserted: the values; that no pattern beats the nominal 8192 FLOP/clk/SM time (N/2 clocks) at N >= 64; that N = 128 runs
at it from one warp and N = 64 from two warps (one warp alone: 44.8 clocks per instruction whatever N -- a per-warp issue
interval); and that the e4m3 instruction (twice the K) never costs more than the fp16 one plus 10 % --
i.e. FP8 operands really would halve the tensor time.  The figures go to BASELINE.md sec. 5 next to the accuracy study
that rules the mode out.  -m gpu."""
import json
import os
import subprocess

import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_e4m3_mma_values_and_rate_against_fp16(tmp_path):
    exe = str(tmp_path / "tcgen05_kind_rate")
    nvcc = os.path.join(os.environ.get("CUDA_HOME", "/usr/local/cuda"), "bin", "nvcc")
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
                           "-I" + os.path.join(ROOT, "paper_2406_17782_b200", "csrc"),
                           os.path.join(ROOT, "tests", "cuda", "tcgen05_kind_rate.cu"), "-o", exe])
    p = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    print(p.stdout.strip())
    assert p.returncode == 0, p.stdout + p.stderr
    r = json.loads(p.stdout.strip().splitlines()[-1])
    assert r["f16"]["values_ok"] and r["e4m3"]["values_ok"]
    for n in (16, 32, 64, 128):
        for pat in ("_chain", "", "_a_smem", "_two_issuers"):
            f16, f8 = r["f16"][f"clk_per_mma_n{n}{pat}"], r["e4m3"][f"clk_per_mma_n{n}{pat}"]
            assert f8 <= 1.1 * f16, (n, pat, f16, f8)                  # twice the K in the same time
            assert f16 >= 0.9 * n / 2, (n, pat, f16)                   # never faster than 128 x n x 16 MAC at 4096 MAC/clk/SM
    assert r["f16"]["clk_per_mma_n128"] <= 1.1 * 64                    # N = 128: nominal rate from one issuing warp
    assert r["f16"]["clk_per_mma_n64_two_issuers"] <= 1.1 * 32         # N = 64: nominal rate needs two issuing warps ...
    assert 1.2 * 32 <= r["f16"]["clk_per_mma_n64"] <= 1.6 * 32         # ... one warp alone issues every 44.8 clocks; a change is news
