"""Pins for the fp64 oracle (oracle/nbsdf_oracle.c) against things other than itself:
hand-computed worked examples, closed forms, invariants, brute force on tiny inputs.
CPU only.  Each test is chosen so that a plausible mistake (dropped bias, wrong concat order,
transposed weight, missing ReLU, wrong log base, wrong frame handedness) fails at least one.
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
from paper_2406_17782_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _q(u=0.3, v=0.6, fp=0.125, m=0, wi=(0.0, 0.6, 0.8), wo=(0.6, 0.0, 0.8)):
    q = np.zeros(1, dtype=oracle.QUERY_DTYPE)
    q["u"], q["v"], q["footprint"], q["material"] = u, v, fp, m
    q["wi"], q["wo"] = wi, wo
    return q


def test_one_hidden_unit_worked_examples():
    g = json.load(open(os.path.join(GOLDEN, "one_hidden_unit.json")))
    Ws = [np.array(w, np.float32) for w in g["W"]]
    bs = [np.array(b, np.float32) for b in g["b"]]
    qq = g["query"]
    q = _q(qq["u"], qq["v"], qq["footprint"], 0, qq["wi"], qq["wo"])
    for case in g["cases"]:
        Z = np.array([[case["z"]]], np.float32)
        out = oracle.eval_queries(Ws, bs, Z, q)[0]
        # inputs 0.6, 0.8, 0.1, ln(e-1) are fp32-rounded before promotion: allow that, nothing more
        np.testing.assert_allclose(out, case["rgb"], rtol=0, atol=3e-7)
    # with fp32-exact inputs (wi, wo, b4 on a binary grid) the agreement is to 1e-14
    Ws[3] = np.array([[0.5, 1, 1, -1, 0.5, 1, 0.25]], np.float32)
    bs[3] = np.array([0.125], np.float32)
    bs[5] = np.array([0, 0, 0], np.float32)
    q = _q(2.25, -0.75, 0.25, 0, (0.0, 0.5, 0.75), (0.5, 0.0, 0.75))
    # h1=.5,h2=.5,feat=1; g1 = .5+0+.5-.75+.25+0+.1875+.125 = .8125; g2 = 2*.8125-.8f
    g2 = 2 * 0.8125 + float(np.float32(-0.8))
    exp = [math.log1p(math.exp(-g2)) + g2, math.log1p(math.exp(-g2)), math.log(2.0)]
    out = oracle.eval_queries(Ws, bs, np.array([[0.5]], np.float32), q)[0]
    np.testing.assert_allclose(out, exp, rtol=0, atol=1e-14)


def test_softplus_closed_form_values():
    g = json.load(open(os.path.join(GOLDEN, "softplus_values.json")))
    for x, y in g["values"]:
        assert oracle.softplus(x) == pytest.approx(y, rel=1e-15, abs=0)
    for x in (0.3, 2.5, 17.0, 33.0):
        assert oracle.softplus(x) - oracle.softplus(-x) == pytest.approx(x, rel=1e-14)


def test_zero_weight_layers():
    rng = np.random.default_rng(11)
    Ws, bs = synth.make_network(rng, 16, 64)
    Z = synth.make_latents(rng, 4, 16)
    q = synth.make_queries(rng, 64, 4)
    # W6 = 0 -> rgb_c = softplus(b6_c) for every query
    W = [w.copy() for w in Ws]; b = [x.copy() for x in bs]
    W[5][:] = 0; b[5][:] = (0.0, 1.0, -1.0)
    out = oracle.eval_queries(W, b, Z, q)
    exp = [0.6931471805599453, 1.3132616875182228, 0.31326168751822286]
    np.testing.assert_allclose(out, np.tile(exp, (64, 1)), rtol=1e-15)
    # W3 = 0 -> output independent of z, uv, footprint (only wi, wo matter)
    W = [w.copy() for w in Ws]; W[2][:] = 0
    q2 = q.copy()
    q2["u"] = rng.random(64); q2["v"] = rng.random(64); q2["footprint"] = 0.5; q2["material"] = 0
    np.testing.assert_array_equal(oracle.eval_queries(W, bs, Z, q), oracle.eval_queries(W, bs, Z, q2))
    # W4 = 0 -> one constant for all queries, computable by hand from b4, W5, b5, W6, b6
    W = [w.copy() for w in Ws]; W[3][:] = 0
    out = oracle.eval_queries(W, bs, Z, q)
    g1 = np.maximum(bs[3].astype(np.float64), 0)
    g2 = np.maximum(W[4].astype(np.float64) @ g1 + bs[4], 0)
    o = W[5].astype(np.float64) @ g2 + bs[5]
    exp = np.log1p(np.exp(o))
    np.testing.assert_allclose(out, np.tile(exp, (64, 1)), rtol=1e-13)


def _naive_affine_chain(Ws, bs, Z, q):
    """Independent brute force for the ReLU-transparent case: batched X.W^T with transposed storage
    and a different loop order (k outermost), pure-Python floats."""
    n = len(q)
    L = Z.shape[1]
    out = []
    for i in range(n):
        x = [float(Z[q["material"][i]][k]) for k in range(L)]
        x += [float(q["u"][i]) % 1.0, float(q["v"][i]) % 1.0, math.log(float(q["footprint"][i]), 2.0)]

        def lin(vec, W, b):
            Wt = [[float(W[o][k]) for o in range(W.shape[0])] for k in range(W.shape[1])]  # [in][out]
            acc = [float(v) for v in b]
            for k in range(len(vec)):          # k outermost
                for o in range(len(acc)):
                    acc[o] += vec[k] * Wt[k][o]
            return acc
        h = lin(lin(lin(x, Ws[0], bs[0]), Ws[1], bs[1]), Ws[2], bs[2])
        y = h + [float(c) for c in q["wi"][i]] + [float(c) for c in q["wo"][i]]
        o = lin(lin(lin(y, Ws[3], bs[3]), Ws[4], bs[4]), Ws[5], bs[5])
        out.append(o)
    return np.array(out)


@pytest.mark.parametrize("L,H,F", [(2, 3, 2), (5, 4, 3), (3, 7, 5)])
def test_relu_transparent_vs_independent_naive_matmul(L, H, F):
    """All weights, biases, latents >= 0, wi/wo in the positive octant, footprint >= 1 (lf >= 0):
    no ReLU clips, so the decoder is an affine chain; pre-softplus outputs must match a separately
    written triple loop.  Catches transposed operands, wrong concat order, dropped bias."""
    rng = np.random.default_rng(100 + L)
    Ws = [rng.uniform(0, 1, s).astype(np.float32) for s in synth.layer_shapes(L, H, F)]
    bs = [rng.uniform(0, 1, s[0]).astype(np.float32) for s in synth.layer_shapes(L, H, F)]
    Z = rng.uniform(0, 1, (3, L)).astype(np.float32)
    n = 12
    q = np.zeros(n, dtype=oracle.QUERY_DTYPE)
    q["u"] = rng.uniform(0, 3, n); q["v"] = rng.uniform(0, 3, n)
    q["footprint"] = rng.uniform(1, 8, n); q["material"] = rng.integers(0, 3, n)
    w = rng.uniform(0.1, 1, (n, 3)); q["wi"] = w / np.linalg.norm(w, axis=1, keepdims=True)
    w = rng.uniform(0.1, 1, (n, 3)); q["wo"] = w / np.linalg.norm(w, axis=1, keepdims=True)
    o = _naive_affine_chain(Ws, bs, Z, q)
    assert (o > 0).all()
    exp = o + np.log1p(np.exp(-o))
    out = oracle.eval_queries(Ws, bs, Z, q)
    np.testing.assert_allclose(out, exp, rtol=1e-12)


def test_relu_is_applied_on_hidden_layers_only():
    """Negate W1 of a ReLU-transparent net: h1 = 0 exactly, so the result equals the net with W1 = 0, b1 = 0;
    and the feature layer is linear: a negative feature must survive (flip W3's sign -> different output)."""
    rng = np.random.default_rng(5)
    L, H, F = 3, 4, 2
    Ws = [rng.uniform(0.1, 1, s).astype(np.float32) for s in synth.layer_shapes(L, H, F)]
    bs = [rng.uniform(0.1, 1, s[0]).astype(np.float32) for s in synth.layer_shapes(L, H, F)]
    Z = rng.uniform(0.1, 1, (1, L)).astype(np.float32)
    q = _q(0.3, 0.6, 2.0)
    Wn = [w.copy() for w in Ws]; bn = [b.copy() for b in bs]
    Wn[0] = -Wn[0]; bn[0] = -bn[0]
    W0 = [w.copy() for w in Ws]; b0 = [b.copy() for b in bs]
    W0[0][:] = 0; b0[0][:] = 0
    np.testing.assert_array_equal(oracle.eval_queries(Wn, bn, Z, q), oracle.eval_queries(W0, b0, Z, q))
    # linear feature: W3 -> -W3, b3 -> -b3 gives feat -> -feat; compensate by negating W4's feat columns
    Wf = [w.copy() for w in Ws]; bf = [b.copy() for b in bs]
    Wf[2] = -Wf[2]; bf[2] = -bf[2]; Wf[3][:, :F] = -Wf[3][:, :F]
    np.testing.assert_allclose(oracle.eval_queries(Wf, bf, Z, q), oracle.eval_queries(Ws, bs, Z, q), rtol=1e-14)


def test_uv_wrap_periodicity_and_range():
    rng = np.random.default_rng(3)
    Ws, bs = synth.make_network(rng, 16, 64)
    Z = synth.make_latents(rng, 1, 16)
    a = oracle.eval_queries(Ws, bs, Z, _q(u=0.25, v=0.5))
    b = oracle.eval_queries(Ws, bs, Z, _q(u=3.25, v=-1.5))
    np.testing.assert_array_equal(a, b)                       # exact in fp32: bit-for-bit
    assert oracle.wrap(-0.25) == 0.75 and oracle.wrap(2.0) == 0.0 and oracle.wrap(0.999) == 0.999
    assert 0.0 <= oracle.wrap(-1e-9) <= 1.0


def test_log_footprint_exact_and_clamped():
    for k in range(-20, 5):
        assert oracle.log_footprint(2.0 ** k) == float(k)
    for bad in (0.0, -1.0, 1e-30):
        assert oracle.log_footprint(bad) == -20.0
    assert oracle.log_footprint(100.0) == 4.0
    assert oracle.log_footprint(3.0) == pytest.approx(math.log(3.0) / math.log(2.0), rel=1e-15)


def _rot(rng):
    a = rng.standard_normal((3, 3))
    qm, r = np.linalg.qr(a)
    qm = qm * np.sign(np.diag(r))
    if np.linalg.det(qm) < 0:
        qm[:, 0] = -qm[:, 0]
    return qm


def test_local_frame_worked_example_and_rotation_invariance():
    # n = (0, .6, .8), t = (1,0,0) -> t^ = (1,0,0), b^ = n x t = (0, .8, -.6); world +z -> (0, -.6, .8)
    np.testing.assert_allclose(oracle.to_local([0, 0.6, 0.8], [1, 0, 0], [0, 0, 1]), [0, -0.6, 0.8], atol=1e-15)
    np.testing.assert_allclose(oracle.to_local([0, 0.6, 0.8], [1, 0, 0], [1, 0, 0]), [1, 0, 0], atol=1e-15)
    # un-normalised n, tangent hint not orthogonal: Gram-Schmidt
    np.testing.assert_allclose(oracle.to_local([0, 0, 2], [3, 0, 5], [1, 2, 3]), [1, 2, 3], atol=1e-15)
    # right-handed: b = n x t;  n=z, t=y -> b = z x y = -x
    np.testing.assert_allclose(oracle.to_local([0, 0, 1], [0, 1, 0], [1, 0, 0]), [0, -1, 0], atol=1e-15)
    # degenerate tangent (parallel to n): k = argmin |n_k| -> e_0 for n = z;  e_1 for n = (1,0,0)... lowest k on ties
    np.testing.assert_allclose(oracle.to_local([0, 0, 1], [0, 0, 3], [1, 2, 3]), [1, 2, 3], atol=1e-15)
    np.testing.assert_allclose(oracle.to_local([1, 0, 0], [2, 0, 0], [1, 2, 3]), [2, 3, 1], atol=1e-15)
    # joint rotation of (n, t, wi, wo) leaves the decoder output unchanged
    rng = np.random.default_rng(8)
    Ws, bs = synth.make_network(rng, 16, 64)
    Z = synth.make_latents(rng, 2, 16)
    q = synth.make_queries(rng, 32, 2)
    fr = synth.make_frames(rng, 32)
    base = oracle.eval_queries(Ws, bs, Z, q, fr)
    R = _rot(rng)
    q2 = q.copy()
    # rotate in float64 then round to fp32: invariance holds to fp32 input rounding
    q2["wi"] = (q["wi"].astype(np.float64) @ R.T); q2["wo"] = (q["wo"].astype(np.float64) @ R.T)
    fr2 = np.concatenate([fr[:, :3].astype(np.float64) @ R.T, fr[:, 3:].astype(np.float64) @ R.T], 1)
    out = oracle.eval_queries(Ws, bs, Z, q2, fr2)
    np.testing.assert_allclose(out, base, rtol=2e-6)
    # identity frame == no frame
    ident = np.tile(np.array([0, 0, 1, 1, 0, 0], np.float32), (32, 1))
    np.testing.assert_allclose(oracle.eval_queries(Ws, bs, Z, q, ident), oracle.eval_queries(Ws, bs, Z, q), rtol=1e-15)


def test_latent_indirection():
    rng = np.random.default_rng(9)
    Ws, bs = synth.make_network(rng, 16, 64)
    Z = synth.make_latents(rng, 8, 16)
    q = synth.make_queries(rng, 200, 8)
    full = oracle.eval_queries(Ws, bs, Z, q)
    for m in range(8):
        sel = q["material"] == m
        qs = q[sel].copy(); qs["material"] = 0
        np.testing.assert_array_equal(full[sel], oracle.eval_queries(Ws, bs, Z[m:m + 1], qs))
    qn = q.copy(); qn["material"][::3] = -1
    out = oracle.eval_queries(Ws, bs, Z, qn)
    assert (out[::3] == 0).all() and (out[1::3] == full[1::3]).all()


def _one_pixel_gbuffer(x=(0.0, 0.0, 0.0), n=(0.0, 0.0, 1.0), t=(1.0, 0.0, 0.0), u=0.3, v=0.6, fp=0.125, m=0,
                       cam=(0.0, 0.0, 1.0)):
    return {"pos_fp": np.array([[*x, fp]], np.float32), "nrm_u": np.array([[*n, u]], np.float32),
            "tan_v": np.array([[*t, v]], np.float32), "material": np.array([m], np.int32),
            "cam_pos": np.array(cam, np.float32)}


def _lights(*rows):
    lt = np.zeros(len(rows), dtype=oracle.LIGHT_DTYPE)
    for i, (ty, vec, rgb, en) in enumerate(rows):
        lt[i]["type"], lt[i]["vec"], lt[i]["rgb"], lt[i]["emit_n"] = ty, vec, rgb, en
    return lt


def test_shading_closed_forms_and_linearity():
    rng = np.random.default_rng(21)
    Ws, bs = synth.make_network(rng, 16, 64)
    Z = synth.make_latents(rng, 2, 16)
    g = _one_pixel_gbuffer()
    up = (0.0, 0.0, 1.0)
    # BSDF for wi = wo = +z (camera straight above, light along n)
    rgb = oracle.eval_queries(Ws, bs, Z, _q(wi=up, wo=up))[0]
    # 1 directional light along n with radiance (2,2,2): pixel = 2 * rgb * cos(0)
    out = oracle.shade_frame(Ws, bs, Z, g, _lights((0, up, (2, 2, 2), (0, 0, 0))))[0]
    np.testing.assert_allclose(out, 2 * rgb, rtol=1e-15)
    # un-normalised direction gives the same
    out = oracle.shade_frame(Ws, bs, Z, g, _lights((0, (0, 0, 5), (2, 2, 2), (0, 0, 0))))[0]
    np.testing.assert_allclose(out, 2 * rgb, rtol=1e-15)
    # point light 2 units straight above, I = (8,8,8), isotropic -> E = 8/4 = 2 -> same pixel
    out = oracle.shade_frame(Ws, bs, Z, g, _lights((1, (0, 0, 2), (8, 8, 8), (0, 0, 0))))[0]
    np.testing.assert_allclose(out, 2 * rgb, rtol=1e-15)
    # emitter cosine: emitter normal tilted 60 deg from the -wi direction -> factor 0.5
    out = oracle.shade_frame(Ws, bs, Z, g, _lights((1, (0, 0, 2), (8, 8, 8), (math.sqrt(0.75), 0, -0.5))))[0]
    np.testing.assert_allclose(out, rgb, rtol=1e-7)
    # emitter facing away, and light below the horizon -> exactly 0
    assert (oracle.shade_frame(Ws, bs, Z, g, _lights((1, (0, 0, 2), (8, 8, 8), (0, 0, 1)))) == 0).all()
    assert (oracle.shade_frame(Ws, bs, Z, g, _lights((0, (0.6, 0, -0.8), (1, 1, 1), (0, 0, 0)))) == 0).all()
    assert (oracle.shade_frame(Ws, bs, Z, g, _lights()) == 0).all()
    # oblique: directional light (0.6, 0, 0.8) with tilted frame; compare with eval on hand-rotated directions
    g2 = _one_pixel_gbuffer(n=(0.0, 0.6, 0.8), x=(0.1, -0.2, 0.0), cam=(0.1, -0.2, 3.0))
    # wo world = +z -> local (0, -.6, .8); wi world = (0,0.6,0.8)=n -> local (0,0,1); cos = 1; E=(1,.5,.25)
    rgb2 = oracle.eval_queries(Ws, bs, Z, _q(wi=(0, 0, 1), wo=(0, -0.6, 0.8)))[0]
    out = oracle.shade_frame(Ws, bs, Z, g2, _lights((0, (0, 0.6, 0.8), (1, 0.5, 0.25), (0, 0, 0))))[0]
    np.testing.assert_allclose(out, rgb2 * np.array([1, 0.5, 0.25]), rtol=1e-6)
    # linearity in the light set, background pixels
    c = synth.config(2, width=24, height=16)
    gb = c["gbuffer"]; gb["material"] = gb["material"].copy(); gb["material"][5] = -1
    lt = c["lights"]
    full = oracle.shade_frame(c["weights"], c["biases"], c["latents"], gb, lt)
    a = oracle.shade_frame(c["weights"], c["biases"], c["latents"], gb, lt[:2])
    b = oracle.shade_frame(c["weights"], c["biases"], c["latents"], gb, lt[2:])
    np.testing.assert_allclose(full, a + b, rtol=1e-14)
    assert (full[5] == 0).all() and (full[4] > 0).all()
    # pixel range argument
    part = oracle.shade_frame(c["weights"], c["biases"], c["latents"], gb, lt, first=100, count=50)
    np.testing.assert_array_equal(part, full[100:150])


def test_frame_equals_eval_on_expanded_queries():
    """shade_frame == sum over lights of eval(query built by hand in numpy fp64) * E * cos."""
    c = synth.config(2, width=16, height=8)
    gb, lt = c["gbuffer"], c["lights"]
    full = oracle.shade_frame(c["weights"], c["biases"], c["latents"], gb, lt)
    npx = 16 * 8
    acc = np.zeros((npx, 3))
    x = gb["pos_fp"][:, :3].astype(np.float64)
    wo = gb["cam_pos"].astype(np.float64)[None] - x
    wo /= np.linalg.norm(wo, axis=1, keepdims=True)
    frames = np.concatenate([gb["nrm_u"][:, :3], gb["tan_v"][:, :3]], 1)
    for l in lt:
        if l["type"] == 0:
            wi = np.tile(l["vec"].astype(np.float64) / np.linalg.norm(l["vec"].astype(np.float64)), (npx, 1))
            E = np.tile(l["rgb"].astype(np.float64), (npx, 1))
        else:
            vv = l["vec"].astype(np.float64)[None] - x
            d2 = (vv * vv).sum(1, keepdims=True)
            wi = vv / np.sqrt(d2)
            E = l["rgb"].astype(np.float64)[None] / d2
        q = np.zeros(npx, dtype=oracle.QUERY_DTYPE)
        q["u"], q["v"], q["footprint"] = gb["nrm_u"][:, 3], gb["tan_v"][:, 3], gb["pos_fp"][:, 3]
        q["material"] = gb["material"]; q["wi"] = wi; q["wo"] = wo      # fp32-rounded world directions
        rgb = oracle.eval_queries(c["weights"], c["biases"], c["latents"], q, frames)
        n = gb["nrm_u"][:, :3].astype(np.float64)
        cos = np.maximum((wi * n).sum(1) / np.linalg.norm(n, axis=1), 0)[:, None]
        acc += rgb * E * cos
    np.testing.assert_allclose(full, acc, rtol=5e-6)


def test_synth_recipe_properties():
    c = synth.config(0)
    q = c["queries"]
    assert len(q) == 4096 and (q["material"] == 0).all()
    assert (q["u"] >= 0).all() and (q["u"] < 1).all()
    lf = np.log2(q["footprint"]); assert lf.min() >= -8 and lf.max() <= 0
    for k in ("wi", "wo"):
        np.testing.assert_allclose(np.linalg.norm(q[k], axis=1), 1, atol=1e-6)
        assert (q[k][:, 2] >= 0).all()
        assert abs(q[k][:, 2].astype(np.float64).mean() - 2 / 3) < 0.02      # E[cos] = 2/3 for cosine weighting
    c1 = synth.config(1, n=1024)
    for w in c1["weights"]:
        assert (w.view(np.uint32) & 0xFFFF == 0).all()                      # bf16-representable
        np.testing.assert_array_equal(synth.round_to_bf16(w), w)
    a = math.sqrt(6 / (19 + 64)); assert abs(c["weights"][0]).max() <= a
    g = synth.config(2, width=192, height=128)["gbuffer"]
    assert g["pos_fp"][0, 3] == np.float32(12 / 128)
    ang = np.degrees(np.arccos(g["nrm_u"][:, 2])); assert ang.max() <= 30.001
    assert set(np.unique(g["material"])) <= set(range(8))
    # round_to_bf16 ties-to-even
    x = np.array([1.0 + 2 ** -8, 1.0 + 3 * 2 ** -8, 1.0 + 2 ** -8 + 2 ** -20], np.float32)
    np.testing.assert_array_equal(synth.round_to_bf16(x), np.array([1.0, 1.0 + 2 ** -6, 1.0 + 2 ** -7], np.float32))
