"""Parity at PIPELINE DEPTH for every (L, H) point, both tensor-core kernels and the paper-structured one.  -m gpu.

The persistent kernels have structurally different tile loops per dims (merged + x in its own TMEM region; merged
with x sharing the A region; the six-layer loop of H = 128; the light loop of nbsdf_shade_frame) and a two-buffer
bulk-copy staging whose phase logic only matters from a warpgroup's THIRD tile on.  A batch of
3 * num_sms * NWG * 128 + 129 queries gives every warpgroup at least three full tiles plus a ragged round; every output
is compared with the fp64 oracle element by element (BASELINE.json configs[4] dims; tolerance north_star's).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2406_17782_b200 import api, synth  # noqa: E402

from test_gpu_parity import Ctx, check  # noqa: E402

HS, LS = [32, 64, 128], [8, 16, 32]

# bf16 operands carry 8-bit significands through four hidden layers; where that cannot hold the max bound (every H = 32
# network and (L 32, H 64): 0.5-1.2e-2, reproduced without the GPU by tests/quant_emulation.py) nbsdf_create rejects the
# mode (test_gpu_parity.py::test_config4_dims asserts the rejection), so those points do not appear here.  Every bf16
# point that IS served is held to the full bound and, in the eval test, to the bf16-rounded emulation as well.
def dims_params(kind):
    from test_gpu_parity import bf16_served
    out = []
    for prec in ("fp16", "bf16"):
        for L in LS:
            for H in HS:
                if prec == "fp16" or bf16_served(L, H):
                    out.append(pytest.param(prec, L, H, id=f"{prec}-{L}-{H}"))
    return out


NWG_EVAL = {32: 6, 64: 4, 128: 2}          # warpgroups per CTA (csrc/nbsdf_tc.cu launch_one); an over-estimate is harmless
NWG_SHADE = {32: 5, 64: 4, 128: 2}


def num_sms():
    return torch.cuda.get_device_properties(0).multi_processor_count


def lights3():
    """directional + point + point with an emitter normal: first / middle / last iteration of the light loop"""
    lt = synth.lights_direct5()[:3].copy()
    lt[2]["emit_n"] = (0.0, 0.6, -0.8)
    return lt


@pytest.mark.parametrize("prec,L,H", dims_params("eval"))
def test_eval_three_rounds_every_dims(prec, L, H):
    n = 3 * num_sms() * NWG_EVAL[H] * 128 + 129
    seed = synth.sweep_seed(1, HS.index(H), LS.index(L))
    cfg = synth.config(4, n=n, L=L, H=H, seed=seed)
    q = cfg["queries"]
    q["material"][11::97] = -1                                   # background rows inside full tiles
    frames = synth.make_frames(np.random.default_rng(seed + 1), n)
    ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], q)
    ref_f = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], q, frames)
    c = Ctx(cfg, prec, L=L, H=H)
    out = c.eval(q)
    out_f = c.eval(q, frames)
    # a second size on the same context: two full rounds minus one query (the last round has an empty tail)
    n2 = 2 * num_sms() * NWG_EVAL[H] * 128 - 1
    out2 = c.eval(q[:n2])
    c.close()
    live = q["material"] >= 0
    assert (out[~live] == 0).all() and (out_f[~live] == 0).all()
    if prec == "bf16":
        # sharper than the 1e-2 bound, and independent of it: against the oracle's forward pass with the SAME operand
        # rounding (tests/quant_emulation.py), what remains is fp32 accumulation order and the rare rounding decision that
        # flips on it (one flipped bf16 activation is 2^-8 relative, so the max stays a max; measured mean 3e-7..4e-7) --
        # a staging or phase slip in the bf16 instantiation would put the MEAN orders of magnitude above this
        import quant_emulation as quant_study
        emu = quant_study.forward(cfg, q[live], quant_study.bf16, quant_study.bf16, quant_study.bf16, merged=H <= 64)
        r = np.abs(out[live] - emu) / np.maximum(np.abs(emu), 1e-6)
        assert r.max() <= 1e-2 and r.mean() <= 1e-5, f"bf16 kernel vs bf16-rounded oracle: max {r.max()} mean {r.mean()}"
    check(out[live], ref[live], prec, f"eval L={L} H={H} n={n}")
    check(out_f[live], ref_f[live], prec, f"eval+frames L={L} H={H} n={n}")
    np.testing.assert_array_equal(out2.view(np.uint32), out[:n2].view(np.uint32))      # position independence


@pytest.mark.parametrize("prec,L,H", dims_params("shade"))
def test_shade_three_rounds_every_dims(prec, L, H):
    npx_min = 3 * num_sms() * NWG_SHADE[H] * 128 + 77
    W = 509                                                     # odd width: rows never align with 128-pixel tiles
    Hh = (npx_min + W - 1) // W
    seed = synth.sweep_seed(2, HS.index(H), LS.index(L))
    cfg = synth.config(4, n=1, L=L, H=H, seed=seed)
    g = synth.make_gbuffer(np.random.default_rng(seed), W, Hh)
    g["material"] = g["material"].copy()
    g["material"][5::131] = -1
    lights = lights3()
    ref = oracle.shade_frame(cfg["weights"], cfg["biases"], cfg["latents"], g, lights)
    c = Ctx(cfg, prec, L=L, H=H)
    out = c.shade(g, lights)
    c.close()
    live = g["material"] >= 0
    assert (out[~live] == 0).all()
    check(out[live], ref[live], prec, f"shade L={L} H={H} {W}x{Hh}")


@pytest.mark.parametrize("L,H", [(16, 64), (32, 128), (8, 32)])
def test_fp32_variant_at_depth(L, H):
    n = 3 * num_sms() * 4 * 128 + 129
    seed = synth.sweep_seed(3, HS.index(H), LS.index(L))
    cfg = synth.config(4, n=n, L=L, H=H, seed=seed)
    frames = synth.make_frames(np.random.default_rng(seed + 1), n)
    ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"], frames)
    c = Ctx(cfg, "fp32", L=L, H=H)
    out = c.eval(cfg["queries"], frames)
    g = synth.make_gbuffer(np.random.default_rng(seed), 509, 150)
    fr = c.shade(g, lights3())
    c.close()
    check(out, ref, "fp32", f"fp32 eval L={L} H={H}")
    check(fr, oracle.shade_frame(cfg["weights"], cfg["biases"], cfg["latents"], g, lights3()), "fp32", f"fp32 shade L={L} H={H}")


@pytest.mark.parametrize("L,H", [(16, 64), (32, 64), (32, 32), (16, 128), (8, 32)])
def test_soak_random_sizes_and_offsets(L, H):
    """Random (n, offset) launches on one context per structural variant, with and without frames: finite results,
    nothing written past n (NaN canary), every output within tolerance of the oracle."""
    rng = np.random.default_rng(2024 + L + H)
    N = 3 * num_sms() * NWG_EVAL[H] * 128 + 4096
    cfg = synth.config(4, n=N, L=L, H=H, seed=synth.sweep_seed(4, HS.index(H), LS.index(L)))
    fr = synth.make_frames(rng, N)
    ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"])
    reff = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"], fr)
    c = Ctx(cfg, "fp16", L=L, H=H)
    qd = api.queries_to_device(cfg["queries"])
    frd = torch.from_numpy(fr).cuda()
    out = torch.empty((N, 3), dtype=torch.float32, device="cuda")
    for it in range(40):
        n = int(rng.integers(1, N))
        off = int(rng.integers(0, (N - n) // 2 + 1)) * 2          # even record offset keeps 16-byte alignment (80 B)
        out.fill_(float("nan"))
        if it % 2 == 0:
            api.nbsdf_eval(c.ctx, qd[off * 40:], None, n, out)
            r = ref[off:off + n]
        else:
            api.nbsdf_eval(c.ctx, qd[off * 40:], frd[off:], n, out)
            r = reff[off:off + n]
        torch.cuda.synchronize()
        got = out[:n].cpu().numpy()
        assert np.isfinite(got).all(), (it, n, off)
        assert torch.isnan(out[n:]).all(), "wrote past n"
        rel = np.abs(got - r) / np.maximum(np.abs(r), 1e-6)
        assert rel.max() <= 1e-2, (it, n, off, rel.max())
    c.close()


def test_soak_paper_decoder():
    rng = np.random.default_rng(99)
    N = 3 * num_sms() * 4 * 128 + 4096
    pc = synth.pd_config("eval", n=N)
    fr = synth.make_frames(rng, N)
    pref = oracle.pd_eval_queries(pc["weights"], pc["biases"], pc["latents"], pc["albedos"], pc["queries"])
    preff = oracle.pd_eval_queries(pc["weights"], pc["biases"], pc["latents"], pc["albedos"], pc["queries"], fr)
    ctx = api.nbsdf_create_paper(pc["weights"], pc["biases"], 64, 8, "fp16")
    api.nbsdf_set_latents(ctx, 0, pc["latents"])
    api.nbsdf_set_albedos(ctx, 0, pc["albedos"])
    qd = api.queries_to_device(pc["queries"])
    frd = torch.from_numpy(fr).cuda()
    out = torch.empty((N, 3), dtype=torch.float32, device="cuda")
    for it in range(30):
        n = int(rng.integers(1, N))
        off = int(rng.integers(0, (N - n) // 2 + 1)) * 2
        out.fill_(float("nan"))
        api.nbsdf_eval(ctx, qd[off * 40:], frd[off:] if it % 2 else None, n, out)
        torch.cuda.synchronize()
        r = (preff if it % 2 else pref)[off:off + n]
        got = out[:n].cpu().numpy()
        assert np.isfinite(got).all() and torch.isnan(out[n:]).all(), (it, n, off)
        rel = np.abs(got - r) / np.maximum(np.abs(r), 1e-6)
        assert rel.max() <= 1e-2, (it, n, off, rel.max())
    api.nbsdf_destroy(ctx)
