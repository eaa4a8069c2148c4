"""Parity of the paper-structured CUDA decoder (nbsdf_create_paper, through the C ABI) against its fp64 oracle.  -m gpu.

Tolerance: the same metric and bounds as the BASELINE.json decoder,
rel = |gpu - ref| / max(|ref|, 1e-6) per channel, max <= 1e-2 and mean <= 2e-3 (north_star), over all outputs of a case.
Operands are fp16.  bf16 operands are REJECTED at nbsdf_create_paper (NBSDF_E_UNSUPPORTED): the specular outputs are
log-mapped, so an ABSOLUTE error d of the raw output o ~ 3 becomes a RELATIVE error d of
S = (e^o - 1)/k, and 8-bit significands through seven layers measured 4e-2 -- outside the bound, so the mode is not shipped.
The synthetic network (synth.make_pd_network) keeps the BSDF values positive and O(1), as a BSDF's are.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2406_17782_b200 import api, synth  # noqa: E402

PRECS = ["fp16"]
TOL = {"fp16": (1e-2, 2e-3)}


def check(gpu, ref, what="", prec="fp16"):
    TMAX, TMEAN = TOL[prec]
    gpu = np.asarray(gpu, np.float64).reshape(-1, 3)
    ref = np.asarray(ref, np.float64).reshape(-1, 3)
    assert np.isfinite(gpu).all(), what
    r = np.abs(gpu - ref) / np.maximum(np.abs(ref), 1e-6)
    mx, mean = r.max(axis=0), r.mean(axis=0)
    assert (mx <= TMAX).all() and (mean <= TMEAN).all(), f"{what}: max {mx} mean {mean}"
    return mx, mean


class PCtx:
    def __init__(self, cfg, prec, M=None):
        M = cfg["latents"].shape[0] if M is None else M
        self.ctx = api.nbsdf_create_paper(cfg["weights"], cfg["biases"], 64, M, prec)
        api.nbsdf_set_latents(self.ctx, 0, cfg["latents"])
        api.nbsdf_set_albedos(self.ctx, 0, cfg["albedos"])

    def eval(self, q, frames=None):
        n = len(q)
        qd = api.queries_to_device(q) if n else None
        fd = torch.from_numpy(np.ascontiguousarray(frames, np.float32)).cuda() if frames is not None and n else None
        out = torch.full((max(n, 1), 3), float("nan"), dtype=torch.float32, device="cuda")
        api.nbsdf_eval(self.ctx, qd, fd, n, out if n else None)
        torch.cuda.synchronize()
        return out[:n].cpu().numpy()

    def shade(self, g, lights):
        gd = api.gbuffer_to_device(g)
        npx = g["width"] * g["height"]
        out = torch.full((npx, 3), float("nan"), dtype=torch.float32, device="cuda")
        api.nbsdf_shade_frame(self.ctx, gd, lights, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def close(self):
        api.nbsdf_destroy(self.ctx)


def _args(cfg):
    return cfg["weights"], cfg["biases"], cfg["latents"], cfg["albedos"]


@pytest.mark.parametrize("prec", PRECS)
def test_paper_eval_small_and_tile_edges(prec):
    cfg = synth.pd_config("eval", n=4096 + 77)
    ref = oracle.pd_eval_queries(*_args(cfg), cfg["queries"])
    c = PCtx(cfg, prec)
    check(c.eval(cfg["queries"]), ref, f"paper eval {prec}", prec)
    outs, refs = [], []
    for n in (0, 1, 127, 128, 129, 1025):
        out = c.eval(cfg["queries"][:n])
        assert out.shape == (n, 3)
        if n:                 # max bound per batch, mean bound on the pooled outputs
            r = np.abs(out - ref[:n]) / np.maximum(np.abs(ref[:n]), 1e-6)
            assert np.isfinite(out).all() and r.max() <= TOL[prec][0], f"paper eval n={n}"
            outs.append(out)
            refs.append(ref[:n])
    check(np.concatenate(outs), np.concatenate(refs), f"paper eval tile edges pooled {prec}", prec)
    c.close()


@pytest.mark.parametrize("prec", PRECS)
def test_paper_frames_background_wrap_and_transmission(prec):
    cfg = synth.pd_config("eval", n=3000, seed=21)
    q = cfg["queries"].copy()
    q["material"][5::37] = -1
    q["u"] += np.float32(3.0)
    q["v"] -= np.float32(2.0)
    q["footprint"][::11] = 7.5           # beyond the clamp
    q["footprint"][1::11] = -1.0
    rng = np.random.default_rng(4)
    frames = synth.make_frames(rng, len(q))
    ref = oracle.pd_eval_queries(*_args(cfg), q, frames=frames)
    c = PCtx(cfg, prec)
    out = c.eval(q, frames)
    assert (out[5::37] == 0).all()
    live = q["material"] >= 0
    check(out[live], ref[live], f"paper frames {prec}", prec)
    # wo.z is not an input: bit-identical when it changes
    q2 = cfg["queries"].copy()
    a = c.eval(q2)
    q2["wo"][:, 2] = 0.123
    np.testing.assert_array_equal(c.eval(q2).view(np.uint32), a.view(np.uint32))
    # batch permutation gives permuted identical bits
    perm = rng.permutation(len(q2))
    np.testing.assert_array_equal(c.eval(cfg["queries"][perm]).view(np.uint32), a[perm].view(np.uint32))
    c.close()


@pytest.mark.parametrize("prec", PRECS)
def test_paper_frame_shading_and_albedo_edit(prec):
    cfg = synth.pd_config("frame", width=320, height=136)
    g = cfg["gbuffer"]
    g["material"] = g["material"].copy(); g["material"][7::53] = -1
    ref = oracle.pd_shade_frame(*_args(cfg), g, cfg["lights"])
    c = PCtx(cfg, prec)
    out = c.shade(g, cfg["lights"])
    assert (out[7::53] == 0).all()
    live = g["material"] >= 0
    check(out[live], ref[live], f"paper frame {prec}", prec)
    assert (c.shade(g, cfg["lights"][:0]) == 0).all()
    # one light only, behind the fabric: transmission contributes (|cos| weighting)
    back = c.shade(g, cfg["lights"][5:6])
    check(back[live], oracle.pd_shade_frame(*_args(cfg), g, cfg["lights"][5:6])[live], f"paper back light {prec}", prec)
    assert (back[live] > 0).all()
    # albedo edit (no network inference involved): only material 3 changes, and it matches the oracle
    A2 = cfg["albedos"].copy()
    A2[3] = np.linspace(0.1, 0.9, 12, dtype=np.float32)
    api.nbsdf_set_albedos(c.ctx, 3, A2[3])
    out2 = c.shade(g, cfg["lights"])
    other = live & (g["material"] != 3)
    np.testing.assert_array_equal(out2[other].view(np.uint32), out[other].view(np.uint32))
    ref2 = oracle.pd_shade_frame(cfg["weights"], cfg["biases"], cfg["latents"], A2, g, cfg["lights"])
    check(out2[live], ref2[live], f"paper albedo edit {prec}", prec)
    c.close()


def test_paper_decoder_with_64_materials():
    """max_materials = 64 on the paper-structured kernel: the padded 64-row latent table and the 64 x 12 albedo table at
    full size, per-pixel-random material ids; every output of a multi-tile batch and of a frame against the oracle."""
    M = 64
    cfg = synth.pd_config("eval", n=148 * 128 * 2 + 91, M=M, seed=64)
    q = cfg["queries"]
    q["material"][:M] = np.arange(M)
    q["material"][M + 1::89] = -1
    c = PCtx(cfg, "fp16", M=M)
    out = c.eval(q)
    fcfg = synth.pd_config("frame", width=301, height=97, M=M, seed=65)
    g, lights = fcfg["gbuffer"], fcfg["lights"]
    g["material"] = np.random.default_rng(66).integers(-1, M, size=301 * 97).astype(np.int32)
    c2 = PCtx(fcfg, "fp16", M=M)
    fr = c2.shade(g, lights)
    c.close()
    c2.close()
    live = q["material"] >= 0
    assert len(np.unique(q["material"])) == M + 1 and (out[~live] == 0).all()
    check(out[live], oracle.pd_eval_queries(*_args(cfg), q)[live], "paper decoder, 64 materials, eval")
    lv = g["material"] >= 0
    assert (fr[~lv] == 0).all()
    check(fr[lv], oracle.pd_shade_frame(*_args(fcfg), g, lights)[lv], "paper decoder, 64 materials, frame")


def test_paper_frame_with_emitter_normals():
    """Point lights with an emitter normal (E = I max(0, -wi . n_e) / d^2), one of them behind the fabric, one facing
    away (contributes exactly 0): pd_kernel's light loop against the oracle."""
    cfg = synth.pd_config("frame", width=333, height=97, seed=31)
    g = cfg["gbuffer"]
    lights = cfg["lights"].copy()
    lights[1]["emit_n"] = (0.0, 0.6, -0.8)
    lights[3]["emit_n"] = (0.0, 0.0, 1.0)           # above the fabric, facing up: black
    lights[5]["emit_n"] = (0.28, 0.0, 0.96)         # behind the fabric, facing it
    ref = oracle.pd_shade_frame(*_args(cfg), g, lights)
    c = PCtx(cfg, "fp16")
    out = c.shade(g, lights)
    check(out, ref, "paper frame, emitter normals")
    only = c.shade(g, lights[3:4])
    assert (only == 0).all()
    c.close()


def test_paper_frame_per_pixel_albedo_plane():
    """Eq. 8 per pixel: albedos from a [h*w][12] plane instead of the material table."""
    cfg = synth.pd_config("frame", width=333, height=97, seed=41)
    g, lights = cfg["gbuffer"], cfg["lights"]
    g["material"] = g["material"].copy()
    g["material"][3::71] = -1
    rng = np.random.default_rng(5)
    npx = g["width"] * g["height"]
    gA = dict(g, albedo=rng.uniform(0.05, 0.95, (npx, 12)).astype(np.float32))
    ref = oracle.pd_shade_frame(*_args(cfg), gA, lights)
    c = PCtx(cfg, "fp16")
    out = c.shade(gA, lights)
    live = g["material"] >= 0
    assert (out[~live] == 0).all()
    check(out[live], ref[live], "paper frame, per-pixel albedos")
    # a plane that repeats every pixel's table row takes the same arithmetic path: identical bits
    gT = dict(g, albedo=cfg["albedos"][np.maximum(g["material"], 0)])
    np.testing.assert_array_equal(c.shade(gT, lights).view(np.uint32), c.shade(g, lights).view(np.uint32))
    c.close()
    # the BASELINE.json decoder has no albedos: a plane is rejected there
    c0 = synth.config(2, width=16, height=8)
    ctx = api.nbsdf_create(c0["weights"], c0["biases"], 16, 64, 8, "fp16")
    g0 = dict(c0["gbuffer"], albedo=np.zeros((128, 12), np.float32))
    with pytest.raises(api.NbsdfError) as e:
        api.nbsdf_shade_frame(ctx, api.gbuffer_to_device(g0), c0["lights"], torch.empty((128, 3), device="cuda"))
    assert e.value.status == api.NBSDF_E_INVALID
    api.nbsdf_destroy(ctx)


def test_paper_frame_matches_eval_on_expanded_queries():
    """The frame kernel runs the fusion layers once per pixel; nbsdf_eval on the (pixel, light) list does not."""
    cfg = synth.pd_config("frame", width=64, height=40)
    g, lights = cfg["gbuffer"], cfg["lights"]
    c = PCtx(cfg, "fp16")
    frame = c.shade(g, lights).astype(np.float64)
    npx = 64 * 40
    x = g["pos_fp"][:, :3].astype(np.float64)
    cam = g["cam_pos"].astype(np.float64)
    wo = cam[None, :] - x
    wo /= np.linalg.norm(wo, axis=1, keepdims=True)
    frames = np.concatenate([g["nrm_u"][:, :3], g["tan_v"][:, :3]], axis=1).astype(np.float32)
    acc = np.zeros((npx, 3))
    for l in range(len(lights)):
        q = np.zeros(npx, dtype=synth.QUERY_DTYPE)
        q["u"], q["v"], q["footprint"], q["material"] = g["nrm_u"][:, 3], g["tan_v"][:, 3], g["pos_fp"][:, 3], g["material"]
        if lights["type"][l] == 0:
            d = lights["vec"][l].astype(np.float64)
            wi = np.tile(d / np.linalg.norm(d), (npx, 1))
            E = np.tile(lights["rgb"][l].astype(np.float64), (npx, 1))
        else:
            v = lights["vec"][l].astype(np.float64)[None, :] - x
            d2 = (v * v).sum(1, keepdims=True)
            wi = v / np.sqrt(d2)
            E = lights["rgb"][l].astype(np.float64)[None, :] / d2
        q["wi"], q["wo"] = wi.astype(np.float32), wo.astype(np.float32)
        f = c.eval(q, frames).astype(np.float64)
        nrm = g["nrm_u"][:, :3].astype(np.float64)
        nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
        acc += f * E * np.abs((wi * nrm).sum(1, keepdims=True))
    c.close()
    np.testing.assert_allclose(frame, acc, rtol=6e-3)


def test_paper_full_size_batch_and_errors():
    cfg = synth.pd_config("eval")                       # 2^20 queries
    ref = oracle.pd_eval_queries(*_args(cfg), cfg["queries"])
    c = PCtx(cfg, "fp16")
    mx, mean = check(c.eval(cfg["queries"]), ref, "paper eval 2^20 fp16")
    print("paper eval 2^20 fp16: max rel", mx, "mean rel", mean)
    c.close()
    # the fp32 CUDA-core variant is not built for this structure and bf16 operands cannot meet the tolerance (see the
    # module docstring): both are rejected, not silently served; BASELINE.json contexts have no albedo table
    for bad in ("fp32", "bf16"):
        with pytest.raises(api.NbsdfError) as e:
            api.nbsdf_create_paper(cfg["weights"], cfg["biases"], 64, 8, bad)
        assert e.value.status == api.NBSDF_E_UNSUPPORTED
    c0 = synth.config(0)
    ctx = api.nbsdf_create(c0["weights"], c0["biases"], 16, 64, 1, "fp16")
    with pytest.raises(api.NbsdfError) as e:
        api.nbsdf_set_albedos(ctx, 0, np.zeros(12, np.float32))
    assert e.value.status == api.NBSDF_E_INVALID
    api.nbsdf_destroy(ctx)
