"""Pins for the paper-structured fp64 oracle (oracle/nbsdf_oracle_paper.c) against things other than itself:
a hand-computed worked example, closed forms, invariants and an independently written brute-force composition.
CPU only.  Chosen so that a plausible mistake (dropped skip connection, wrong slope, wrong k, wrong concat order,
wo.z leaking in, transposed albedo table, one-blob bin offset) fails at least one.
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
from paper_2406_17782_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _q(u=0.3, v=0.6, size=0.7, m=0, wi=(0.0, 0.6, 0.8), wo=(0.6, 0.0, 0.8)):
    q = np.zeros(1, dtype=oracle.QUERY_DTYPE)
    q["u"], q["v"], q["footprint"], q["material"] = u, v, size, m
    q["wi"], q["wo"] = wi, wo
    return q


def _small_net(rng, L=3, H=5, F=2, lo=-1.0, hi=1.0):
    shapes = synth.pd_layer_shapes(L, H, F)
    Ws = [rng.uniform(lo, hi, s).astype(np.float32) for s in shapes]
    bs = [rng.uniform(lo, hi, s[0]).astype(np.float32) * np.float32(0.1) for s in shapes]
    return Ws, bs


# ---------------------------------------------------------------------------------------------------
def test_oneblob_closed_form():
    """PAPER.md:164 '3 to 24 channels' = 8 bins per scalar; Gaussian of sigma 1/k sampled at bin centres (reading)."""
    k = 8
    # s on a bin centre: entries are exp(-d^2/2) for the integer bin distance d
    for j in range(k):
        got = oracle.oneblob((j + 0.5) / k, k)
        want = [math.exp(-0.5 * (i - j) ** 2) for i in range(k)]
        np.testing.assert_allclose(got, want, rtol=1e-14)
    # s = 0: half-integer distances
    np.testing.assert_allclose(oracle.oneblob(0.0, k), [math.exp(-0.5 * (i + 0.5) ** 2) for i in range(k)], rtol=1e-14)
    # mirror symmetry
    for s in (0.1, 0.37, 0.93):
        np.testing.assert_allclose(oracle.oneblob(s, k), oracle.oneblob(1.0 - s, k)[::-1], rtol=1e-12)
    # the blob peaks in the bin that contains s
    for s in (0.01, 0.26, 0.74, 0.99):
        assert int(np.argmax(oracle.oneblob(s, k))) == int(s * k)


def test_scalar_helpers():
    assert oracle.leaky(3.0) == 3.0 and oracle.leaky(0.0) == 0.0
    assert oracle.leaky(-2.0) == pytest.approx(-0.02, abs=1e-17)
    assert oracle.size01(-1.0) == 0.0 and oracle.size01(0.0) == 0.0
    assert oracle.size01(2.5) == 0.5 and oracle.size01(5.0) == 1.0 and oracle.size01(7.0) == 1.0
    # g(x) = ln(k x + 1), PAPER.md:172-177 (Eq. 9); the oracle applies its inverse
    for k in (100.0, 1000.0):
        for S in (0.0, 1e-4, 0.03, 1.0, 25.0):
            assert oracle.inv_logmap(math.log(k * S + 1.0), k) == pytest.approx(S, rel=1e-12, abs=1e-18)
    assert oracle.inv_logmap(math.log(101.0), 100.0) == pytest.approx(1.0, rel=1e-14)
    assert oracle.inv_logmap(1e-9, 100.0) == pytest.approx(1e-11, rel=1e-8)      # expm1, not exp - 1


def test_one_hidden_unit_worked_example():
    g = json.load(open(os.path.join(GOLDEN, "paper_one_hidden_unit.json")))
    net = g["network"]
    W1 = np.zeros((1, 25), np.float32)
    W1[0, 0] = net["W1_nonzero"]["z"]
    W1[0, 1 + 2] = net["W1_nonzero"]["blob_u[2]"]
    W1[0, 1 + 8 + 4] = net["W1_nonzero"]["blob_v[4]"]
    W1[0, 1 + 16 + 2] = net["W1_nonzero"]["blob_size[2]"]
    Ws = [W1, np.array([[net["W2"]]], np.float32), np.array([net["W3"]], np.float32),
          np.array([[net["W4"]]], np.float32), np.array([[net["W5"]]], np.float32),
          np.array([[net["W6"]]], np.float32), np.array(net["W7"], np.float32).reshape(4, 1)]
    bs = [np.array([net["b1"]], np.float32), np.array([net["b2"]], np.float32), np.array([net["b3"]], np.float32),
          np.array([net["b4"]], np.float32), np.array([net["b5"]], np.float32), np.array([net["b6"]], np.float32),
          np.array(net["b7"], np.float32)]
    Z = np.array([[g["latent"]]], np.float32)
    A = np.array([g["albedo"]], np.float32)
    qq = g["query"]
    for case in g["cases"]:
        q = _q(qq["u"], qq["v"], qq["size"], 0, case["wi"], qq["wo"])
        rgb, comp = oracle.pd_eval_queries(Ws, bs, Z, A, q, components=True)
        # 0.6, 0.8, 0.1, 0.4, ln 101 are fp32-rounded before promotion: allow that (amplified by |W7| = 50), no more
        np.testing.assert_allclose(comp[0], case["components"], rtol=0, atol=2e-6)
        np.testing.assert_allclose(rgb[0], case["rgb"], rtol=0, atol=2e-5)


def test_zero_output_layer_gives_bias_components():
    rng = np.random.default_rng(5)
    Ws, bs = _small_net(rng)
    Ws[6][:] = 0.0
    bs[6][:] = np.array([0.3, 0.7, math.log(101.0), math.log(51.0)], np.float32)
    Z = rng.standard_normal((2, 3)).astype(np.float32)
    A = np.zeros((2, 12), np.float32)
    A[1] = np.arange(12)
    S2 = math.expm1(float(np.float32(math.log(101.0)))) / 100.0
    S3 = math.expm1(float(np.float32(math.log(51.0)))) / 100.0
    rgb, comp = oracle.pd_eval_queries(Ws, bs, Z, A, _q(m=1), components=True)
    np.testing.assert_allclose(comp[0], [float(np.float32(0.3)), float(np.float32(0.7)), S2, S3], rtol=1e-13)
    # Eq. 8 with the albedo table laid out [kd_warp, kd_weft, ks_warp, ks_weft] x RGB
    want = [A[1, c] * comp[0, 0] + A[1, 3 + c] * comp[0, 1] + A[1, 6 + c] * comp[0, 2] + A[1, 9 + c] * comp[0, 3]
            for c in range(3)]
    np.testing.assert_allclose(rgb[0], want, rtol=1e-13)
    # transmission side switches k to 1000: same outputs, specular exactly 10x smaller
    _, compT = oracle.pd_eval_queries(Ws, bs, Z, A, _q(m=1, wi=(0.0, 0.6, -0.8)), components=True)
    np.testing.assert_allclose(compT[0, :2], comp[0, :2], rtol=1e-15)
    np.testing.assert_allclose(compT[0, 2:] * 10.0, comp[0, 2:], rtol=1e-14)


def test_basis_albedos_extract_each_component():
    rng = np.random.default_rng(6)
    Ws, bs = _small_net(rng)
    Z = rng.standard_normal((1, 3)).astype(np.float32)
    q = _q()
    _, comp = oracle.pd_eval_queries(Ws, bs, Z, np.zeros((1, 12), np.float32), q, components=True)
    for j in range(4):
        for c in range(3):
            A = np.zeros((1, 12), np.float32)
            A[0, 3 * j + c] = 1.0
            rgb = oracle.pd_eval_queries(Ws, bs, Z, A, q)[0]
            want = np.zeros(3)
            want[c] = comp[0, j]
            np.testing.assert_array_equal(rgb, want)


def _brute_affine(Ws, bs, z, blob24, wi, wo):
    """Independent composition for the case where no leaky ReLU clips (all pre-activations > 0): the network is then
    affine, o = W7 W6 ((W5 W4 + I) d1 + W5 b4 + b5) ..., written with column-major loops over TRANSPOSED weights."""
    def mv(W, b, x):
        Wt = [[float(W[o][i]) for o in range(len(W))] for i in range(len(W[0]))]      # [in][out]
        y = [float(v) for v in b]
        for i in range(len(Wt)):
            for o in range(len(y)):
                y[o] += Wt[i][o] * x[i]
        return y
    x = [float(v) for v in z] + [float(v) for v in blob24]
    a1 = mv(Ws[0], bs[0], x)
    feat = mv(Ws[1], bs[1], a1)
    y = feat + [wi[0], wi[1], wi[2], wo[0], wo[1]]
    d1 = mv(Ws[2], bs[2], y)
    r = mv(Ws[3], bs[3], d1)
    t = mv(Ws[4], bs[4], r)
    d3 = [t[i] + d1[i] for i in range(len(t))]          # the skip connection
    d4 = mv(Ws[5], bs[5], d3)
    return mv(Ws[6], bs[6], d4), (a1, feat, d1, r, d3, d4)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_no_clip_case_matches_independent_affine_composition(seed):
    """All weights, biases, latents >= 0 and directions in the positive octant: every pre-activation is positive, the
    leaky ReLUs are transparent and the decoder is the affine map above (skip connection included)."""
    rng = np.random.default_rng(100 + seed)
    L, H, F = 4, 6, 3
    Ws, bs = _small_net(rng, L, H, F, lo=0.0, hi=0.5)
    Z = rng.uniform(0.0, 1.0, (2, L)).astype(np.float32)
    A = np.zeros((2, 12), np.float32)
    for i in range(8):
        u, v, size = float(rng.random()), float(rng.random()), float(rng.uniform(0, 5))
        wi = rng.uniform(0.1, 0.6, 3).astype(np.float32)
        wo = rng.uniform(0.1, 0.6, 3).astype(np.float32)
        m = int(rng.integers(0, 2))
        q = _q(u, v, size, m, wi, wo)
        qf = q[0]
        blob = np.concatenate([oracle.oneblob(float(qf["u"]), 8), oracle.oneblob(float(qf["v"]), 8),
                               oracle.oneblob(float(qf["footprint"]) / 5.0, 8)])
        o, acts = _brute_affine(Ws, bs, Z[m], blob, [float(x) for x in wi], [float(x) for x in wo])
        assert all(min(a) > 0 for a in acts)
        _, comp = oracle.pd_eval_queries(Ws, bs, Z, A, q, components=True)
        want = [o[0], o[1], math.expm1(o[2]) / 100.0, math.expm1(o[3]) / 100.0]
        np.testing.assert_allclose(comp[0], want, rtol=1e-12)


def test_all_negative_block_scales_by_the_slope():
    """Slope pin: H = 1 chain with every pre-activation negative: each leaky ReLU multiplies by exactly 0.01."""
    W = lambda v: np.array([[v]], np.float32)
    Ws = [np.zeros((1, 25), np.float32), W(1.0), np.zeros((1, 6), np.float32), W(1.0), W(1.0), W(1.0),
          np.array([[1.0], [0.0], [0.0], [0.0]], np.float32)]
    Ws[2][0, 0] = 1.0
    bs = [np.array([-8.0], np.float32)] + [np.zeros(1, np.float32)] * 5 + [np.zeros(4, np.float32)]
    # a1 = -0.08; feat = -0.0008; d1 = -8e-6; r = -8e-8; d3 = lrelu(-8e-8 - 8e-6) = -8.08e-8; d4 = -8.08e-10
    _, comp = oracle.pd_eval_queries(Ws, bs, np.zeros((1, 1), np.float32), np.zeros((1, 12), np.float32), _q(),
                                     components=True)
    assert comp[0, 0] == pytest.approx(-8.08e-10, rel=1e-12)


def test_invariants():
    rng = np.random.default_rng(7)
    cfg = synth.pd_config("eval", n=64, seed=3)
    args = (cfg["weights"], cfg["biases"], cfg["latents"], cfg["albedos"])
    q = cfg["queries"].copy()
    base = oracle.pd_eval_queries(*args, q)
    # pattern periodicity: integer shifts that are exact in fp32 change nothing, bit for bit
    q2 = q.copy()
    q2["u"] = (np.round(q["u"] * 64) / 64).astype(np.float32)
    ref = oracle.pd_eval_queries(*args, q2)
    q2["u"] += np.float32(3.0)
    np.testing.assert_array_equal(oracle.pd_eval_queries(*args, q2), ref)
    # the view direction enters with two channels only: wo.z is ignored
    q3 = q.copy()
    q3["wo"][:, 2] = rng.random(len(q)).astype(np.float32)
    np.testing.assert_array_equal(oracle.pd_eval_queries(*args, q3), base)
    # but wi.z is an input
    q4 = q.copy()
    q4["wi"][:, 2] *= np.float32(0.5)
    assert np.abs(oracle.pd_eval_queries(*args, q4) - base).max() > 1e-4
    # size saturates at 5 pattern lengths
    q5, q6 = q.copy(), q.copy()
    q5["footprint"], q6["footprint"] = 5.0, 9.0
    np.testing.assert_array_equal(oracle.pd_eval_queries(*args, q5), oracle.pd_eval_queries(*args, q6))
    # Eq. 8 is linear in the albedos
    A2 = (cfg["albedos"] * np.float32(2.0)).astype(np.float32)
    np.testing.assert_allclose(oracle.pd_eval_queries(args[0], args[1], args[2], A2, q), 2.0 * base, rtol=1e-14)
    # latent indirection and joint rotation of (n, t, wi, wo)
    m = int(q["material"][5])
    one = q[5:6].copy(); one["material"] = 0
    np.testing.assert_array_equal(
        oracle.pd_eval_queries(args[0], args[1], cfg["latents"][m:m + 1], cfg["albedos"][m:m + 1], one)[0], base[5])
    nrm = np.array([0.0, 0.6, 0.8]); tan = np.array([1.0, 0.0, 0.0]); bit = np.cross(nrm, tan)
    R = np.stack([tan, bit, nrm], axis=1)          # local -> world
    qw = q.copy()
    qw["wi"] = (q["wi"].astype(np.float64) @ R.T).astype(np.float32)
    qw["wo"] = (q["wo"].astype(np.float64) @ R.T).astype(np.float32)
    frames = np.tile(np.concatenate([nrm, tan]).astype(np.float32), (len(q), 1))
    np.testing.assert_allclose(oracle.pd_eval_queries(*args, qw, frames=frames), base, rtol=2e-5)


def test_frame_shading_closed_forms():
    cfg = synth.pd_config("frame", width=8, height=4, seed=9)
    args = (cfg["weights"], cfg["biases"], cfg["latents"], cfg["albedos"])
    g = cfg["gbuffer"]
    npx = 32
    # flat geometry: normal +z, tangent +x, so world == local
    g["nrm_u"][:, :3] = (0.0, 0.0, 1.0)
    lt = np.zeros(3, dtype=oracle.LIGHT_DTYPE)
    lt["type"] = (0, 1, 1)
    lt["vec"] = ((0.0, 0.0, 2.0), (0.1, 0.2, 2.0), (0.3, -0.2, -1.5))      # the third one is BEHIND the fabric
    lt["rgb"] = ((2.0, 2.0, 2.0), (8.0, 4.0, 2.0), (3.0, 3.0, 3.0))
    full = oracle.pd_shade_frame(*args, g, lt)
    # linearity in the light set
    parts = sum(oracle.pd_shade_frame(*args, g, lt[i:i + 1]) for i in range(3))
    np.testing.assert_allclose(full, parts, rtol=1e-13)
    # frame == sum over hand-expanded (pixel, light) queries of f * E * |cos|; |cos| lets transmission through
    cam = g["cam_pos"].astype(np.float64)
    want = np.zeros((npx, 3))
    for l in range(3):
        q = np.zeros(npx, dtype=oracle.QUERY_DTYPE)
        x = g["pos_fp"][:, :3].astype(np.float64)
        q["u"], q["v"], q["footprint"], q["material"] = g["nrm_u"][:, 3], g["tan_v"][:, 3], g["pos_fp"][:, 3], g["material"]
        wo = cam[None, :] - x
        wo /= np.linalg.norm(wo, axis=1, keepdims=True)
        if lt["type"][l] == 0:
            wi = np.tile(lt["vec"][l].astype(np.float64) / np.linalg.norm(lt["vec"][l].astype(np.float64)), (npx, 1))
            E = np.tile(lt["rgb"][l].astype(np.float64), (npx, 1))
        else:
            v = lt["vec"][l].astype(np.float64)[None, :] - x
            d2 = (v * v).sum(1, keepdims=True)
            wi = v / np.sqrt(d2)
            E = lt["rgb"][l].astype(np.float64)[None, :] / d2
        q["wi"], q["wo"] = wi.astype(np.float32), wo.astype(np.float32)
        f = oracle.pd_eval_queries(*args, q)
        want += f * E * np.abs(wi[:, 2:3])
    np.testing.assert_allclose(full, want, rtol=3e-6)     # wi, wo pass through fp32 in the expanded path
    assert (np.abs(oracle.pd_shade_frame(*args, g, lt[2:3])) > 0).all()
    # background pixels are exactly zero
    g["material"][3] = -1
    assert (oracle.pd_shade_frame(*args, g, lt)[3] == 0).all()


def test_frame_shading_emitter_cosine_closed_form():
    """The emit_n != 0 branch of oracle_pd_shade_frame: E = I max(0, -wi . n_e) / d^2.  With one
    point light, the frame with an emitter normal equals the isotropic frame times max(0, -wi . n_e) pixel by pixel, the
    factor computed here from the geometry alone; a light facing away gives exactly 0; a hand example: pixel at the
    origin, light at (0, 0, 2), n_e = (0, 0.6, -0.8) => factor 0.8."""
    cfg = synth.pd_config("frame", width=8, height=4, seed=10)
    args = (cfg["weights"], cfg["biases"], cfg["latents"], cfg["albedos"])
    g = cfg["gbuffer"]
    x = g["pos_fp"][:, :3].astype(np.float64)
    for pos, en in (((0.3, -0.2, 1.5), (0.0, 0.6, -0.8)), ((0.1, 0.4, -0.9), (0.6, 0.0, 0.8))):   # above / BEHIND the fabric
        lt = np.zeros(1, dtype=oracle.LIGHT_DTYPE)
        lt["type"], lt["vec"], lt["rgb"] = 1, pos, (3.0, 2.0, 1.0)
        iso = oracle.pd_shade_frame(*args, g, lt)
        lt["emit_n"] = en
        got = oracle.pd_shade_frame(*args, g, lt)
        v = np.array(pos, np.float32).astype(np.float64)[None, :] - x
        wi = v / np.linalg.norm(v, axis=1, keepdims=True)
        fac = np.maximum(0.0, -(wi * np.array(en, np.float32).astype(np.float64)[None, :]).sum(1, keepdims=True))
        assert (fac > 0).all() and (np.abs(iso) > 0).all()
        np.testing.assert_allclose(got, iso * fac, rtol=1e-13)
        lt["emit_n"] = tuple(-c for c in en)                                   # emitter facing away: exactly black
        assert (oracle.pd_shade_frame(*args, g, lt) == 0).all()
    g["pos_fp"][0, :3] = 0.0
    lt = np.zeros(1, dtype=oracle.LIGHT_DTYPE)
    lt["type"], lt["vec"], lt["rgb"] = 1, (0.0, 0.0, 2.0), (3.0, 2.0, 1.0)
    iso = oracle.pd_shade_frame(*args, g, lt, first=0, count=1)
    lt["emit_n"] = (0.0, 0.6, -0.8)
    np.testing.assert_allclose(oracle.pd_shade_frame(*args, g, lt, first=0, count=1), iso * np.float64(np.float32(0.8)), rtol=1e-13)


def test_per_pixel_albedo_plane():
    """PAPER.md:261 / Eq. 8 per pixel: a plane that repeats each pixel's material row reproduces the table path bit for
    bit; a basis plane extracts one component per pixel; the frame is linear in the plane; the table is ignored when a
    plane is given."""
    cfg = synth.pd_config("frame", width=8, height=4, seed=13)
    args = (cfg["weights"], cfg["biases"], cfg["latents"])
    g, lt = dict(cfg["gbuffer"]), cfg["lights"]
    base = oracle.pd_shade_frame(*args, cfg["albedos"], g, lt)
    g["albedo"] = cfg["albedos"][g["material"]]
    np.testing.assert_array_equal(oracle.pd_shade_frame(*args, cfg["albedos"], g, lt), base)
    np.testing.assert_array_equal(oracle.pd_shade_frame(*args, np.zeros_like(cfg["albedos"]), g, lt), base)   # table unused
    rng = np.random.default_rng(2)
    A1 = rng.uniform(0.1, 0.9, (32, 12)).astype(np.float32)
    A2 = rng.uniform(0.1, 0.9, (32, 12)).astype(np.float32)
    f = lambda A: oracle.pd_shade_frame(*args, cfg["albedos"], dict(g, albedo=A), lt)          # noqa: E731
    np.testing.assert_allclose(f(A1.astype(np.float64) + A2), f(A1) + f(A2), rtol=2e-7)          # fp32 storage of the sum
    # pixel 5 gets kd_warp = (1, 0, 0) and nothing else: its red channel is sum_l C_warp E_r |cos|, green and blue vanish
    B = np.zeros((32, 12), np.float32)
    B[5, 0] = 1.0
    out = f(B)
    assert out[5, 0] > 0 and out[5, 1] == 0 and out[5, 2] == 0 and (np.delete(out, 5, 0) == 0).all()
    g["material"] = g["material"].copy()
    g["material"][5] = -1
    assert (oracle.pd_shade_frame(*args, cfg["albedos"], dict(g, albedo=B), lt)[5] == 0).all()   # background stays black


def test_lerp_latent_closed_forms():
    """interpolation and extrapolation of two material latent vectors."""
    za = np.array([1.0, -2.0, 0.5, 8.0], np.float32)
    zb = np.array([3.0, 2.0, 0.5, -8.0], np.float32)
    np.testing.assert_array_equal(oracle.lerp_latent(za, zb, 0.0), za.astype(np.float64))
    np.testing.assert_array_equal(oracle.lerp_latent(za, zb, 1.0), zb.astype(np.float64))
    np.testing.assert_array_equal(oracle.lerp_latent(za, zb, 0.5), [2.0, 0.0, 0.5, 0.0])
    np.testing.assert_array_equal(oracle.lerp_latent(za, zb, 0.25), [1.5, -1.0, 0.5, 4.0])
    np.testing.assert_array_equal(oracle.lerp_latent(za, zb, 1.5), [4.0, 4.0, 0.5, -16.0])      # extrapolation
    np.testing.assert_array_equal(oracle.lerp_latent(za, zb, -0.5), [0.0, -4.0, 0.5, 16.0])
