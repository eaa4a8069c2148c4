"""Seeded synthetic inputs for the decoder hot path -- data only, none of the method's arithmetic.

These inputs stand in for the paper's four Falcor scenes, its trained 64-d latents and its
1920x1080 single-light workload, none of which are available.
Shapes and ranges follow BASELINE.json ``configs`` (which echo Table 2, PAPER.md:210-220:
position in (0,1)^2 of the pattern, footprint from sub-period to multi-period, directions over
the hemisphere).  The recipe and draw order are documented in DESIGN.md "Input recipe".

Served to both the oracle (via tests/bench) and the CUDA path; imports neither.
Everything is numpy; one ``numpy.random.default_rng(seed)`` per config, fixed draw order.
"""
import math

import numpy as np

QUERY_DTYPE = np.dtype([("u", "<f4"), ("v", "<f4"), ("footprint", "<f4"), ("material", "<i4"),
                        ("wi", "<f4", (3,)), ("wo", "<f4", (3,))], align=False)
LIGHT_DTYPE = np.dtype([("type", "<i4"), ("vec", "<f4", (3,)), ("rgb", "<f4", (3,)),
                        ("emit_n", "<f4", (3,))], align=False)
FEAT_DIM = 32


def round_to_bf16(a):
    """fp32 -> nearest bf16-representable fp32 (round to nearest even on the dropped 16 bits).
    'Weights stored in bf16' (BASELINE.json configs[1]): the stored values ARE the model, and both
    the oracle and the CUDA library are handed these already-rounded fp32 arrays."""
    x = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32).astype(np.uint64)
    lsb = (x >> 16) & 1
    r = ((x + 0x7FFF + lsb) >> 16) << 16
    return r.astype(np.uint32).view(np.float32).reshape(np.shape(a))


def layer_shapes(L, H, F=FEAT_DIM):
    return [(H, L + 3), (H, H), (F, H), (H, F + 6), (H, H), (3, H)]


def make_network(rng, L=16, H=64, F=FEAT_DIM, bf16_weights=False):
    """Xavier-uniform weights (gain 1), biases 0.01*N(0,1), fp32.  Draw order: W1,b1,...,W6,b6."""
    Ws, bs = [], []
    for (n_out, n_in) in layer_shapes(L, H, F):
        a = math.sqrt(6.0 / (n_in + n_out))
        W = rng.uniform(-a, a, size=(n_out, n_in)).astype(np.float32)
        b = (0.01 * rng.standard_normal(n_out)).astype(np.float32)
        Ws.append(round_to_bf16(W) if bf16_weights else W)
        bs.append(b)
    return Ws, bs


def make_latents(rng, M, L):
    return rng.standard_normal((M, L)).astype(np.float32)


def cosine_hemisphere(rng, n):
    """r = sqrt(xi1), phi = 2 pi xi2, w = (r cos phi, r sin phi, sqrt(1 - xi1))."""
    xi1 = rng.random(n)
    xi2 = rng.random(n)
    r = np.sqrt(xi1)
    phi = 2.0 * np.pi * xi2
    return np.stack([r * np.cos(phi), r * np.sin(phi), np.sqrt(1.0 - xi1)], axis=1).astype(np.float32)


def make_queries(rng, n, M):
    """Draw order: u, v, log2 fp, wi, wo, material."""
    q = np.zeros(n, dtype=QUERY_DTYPE)
    q["u"] = rng.random(n).astype(np.float32)
    q["v"] = rng.random(n).astype(np.float32)
    q["footprint"] = np.exp2(rng.uniform(-8.0, 0.0, n)).astype(np.float32)
    q["wi"] = cosine_hemisphere(rng, n)
    q["wo"] = cosine_hemisphere(rng, n)
    q["material"] = rng.integers(0, M, n).astype(np.int32) if M > 1 else 0
    return q


def make_frames(rng, n):
    """Per-query world frames [n][6] = (n, t): random unit normal, random non-parallel tangent hint."""
    nrm = rng.standard_normal((n, 3))
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    tan = rng.standard_normal((n, 3))
    return np.concatenate([nrm, tan], axis=1).astype(np.float32)


def make_gbuffer(rng, width, height, uv_scale=12.0, n_ids=8, tile=64):
    """Plane z=0 seen by a pinhole at (0,0,1) looking -z, vertical FOV 60 deg, ray through (px+1/2, py+1/2).
    uv = uv_scale * ((px+1/2)/W, (py+1/2)/H) (left unwrapped -- the library wraps);
    footprint = max(|duv/dx|, |duv/dy|) = uv_scale / H (analytic screen-space derivative);
    normal tilted a ~ U[0, 30 deg] about +z at azimuth phi ~ U[0, 2 pi); tangent hint (1,0,0);
    material = ((px>>6) + (py>>6)) mod n_ids.  Draw order: a, phi."""
    W, H = int(width), int(height)
    px = (np.arange(W, dtype=np.float64) + 0.5)[None, :].repeat(H, 0)
    py = (np.arange(H, dtype=np.float64) + 0.5)[:, None].repeat(W, 1)
    th = math.tan(math.radians(30.0))
    x = (2.0 * px / W - 1.0) * (W / H) * th
    y = (1.0 - 2.0 * py / H) * th
    npx = W * H
    a = rng.uniform(0.0, math.radians(30.0), npx)
    phi = rng.uniform(0.0, 2.0 * np.pi, npx)
    pos_fp = np.empty((npx, 4), np.float32)
    pos_fp[:, 0] = x.reshape(-1)
    pos_fp[:, 1] = y.reshape(-1)
    pos_fp[:, 2] = 0.0
    pos_fp[:, 3] = max(uv_scale / W, uv_scale / H)
    nrm_u = np.empty((npx, 4), np.float32)
    nrm_u[:, 0] = np.sin(a) * np.cos(phi)
    nrm_u[:, 1] = np.sin(a) * np.sin(phi)
    nrm_u[:, 2] = np.cos(a)
    nrm_u[:, 3] = (uv_scale * px / W).reshape(-1)
    tan_v = np.empty((npx, 4), np.float32)
    tan_v[:, 0] = 1.0
    tan_v[:, 1] = 0.0
    tan_v[:, 2] = 0.0
    tan_v[:, 3] = (uv_scale * py / H).reshape(-1)
    ix = (np.arange(W) // tile)[None, :]
    iy = (np.arange(H) // tile)[:, None]
    material = ((ix + iy) % n_ids).astype(np.int32).reshape(-1)
    return {"pos_fp": pos_fp, "nrm_u": nrm_u, "tan_v": tan_v, "material": material,
            "width": W, "height": H, "cam_pos": np.array([0.0, 0.0, 1.0], np.float32)}


def lights_direct5():
    """configs[2]: 1 directional light toward (0.3,0.2,1)/|.| with radiance (1,1,1), plus 4 point
    lights at (+-0.6, +-0.35, 0.5) with distinct RGB intensities ~0.5."""
    lt = np.zeros(5, dtype=LIGHT_DTYPE)
    d = np.array([0.3, 0.2, 1.0])
    lt[0]["type"] = 0
    lt[0]["vec"] = (d / np.linalg.norm(d)).astype(np.float32)
    lt[0]["rgb"] = (1.0, 1.0, 1.0)
    inten = [(0.6, 0.5, 0.4), (0.4, 0.5, 0.6), (0.5, 0.6, 0.4), (0.5, 0.4, 0.6)]
    k = 1
    for sx in (-1.0, 1.0):
        for sy in (-1.0, 1.0):
            lt[k]["type"] = 1
            lt[k]["vec"] = (0.6 * sx, 0.35 * sy, 0.5)
            lt[k]["rgb"] = inten[k - 1]
            k += 1
    return lt


def lights_area16(rng, side=0.5, z=0.8, Le=8.0):
    """configs[3]: one side x side emitter at height z facing -z, sampled at 4x4 jittered strata and
    passed as 16 point lights with rgb = Le*A/16 and emit_n = (0,0,-1); the same 16 samples serve
    every pixel (no RNG inside either implementation).  Draw order: jitter x (16), jitter y (16)."""
    jx = rng.random(16)
    jy = rng.random(16)
    lt = np.zeros(16, dtype=LIGHT_DTYPE)
    for s in range(16):
        i, j = s % 4, s // 4
        lt[s]["type"] = 1
        lt[s]["vec"] = ((-0.5 + (i + jx[s]) / 4.0) * side, (-0.5 + (j + jy[s]) / 4.0) * side, z)
        lt[s]["rgb"] = (Le * side * side / 16.0,) * 3
        lt[s]["emit_n"] = (0.0, 0.0, -1.0)
    return lt


def sweep_seed(i_n, i_h, i_l):
    return 1000 + 9 * i_n + 3 * i_h + i_l


def config(idx, n=None, width=None, height=None, L=16, H=64, seed=None):
    """The five BASELINE.json configs as dicts of numpy arrays.  seed defaults to the config index."""
    rng = np.random.default_rng(idx if seed is None else seed)
    if idx == 0:
        Ws, bs = make_network(rng, L, H)
        Z = make_latents(rng, 1, L)
        q = make_queries(rng, 4096 if n is None else n, 1)
        return {"name": "tiny_eval", "weights": Ws, "biases": bs, "latents": Z, "queries": q}
    if idx in (1, 4):
        Ws, bs = make_network(rng, L, H, bf16_weights=True)
        Z = make_latents(rng, 8, L)
        q = make_queries(rng, (1 << 20) if n is None else n, 8)
        return {"name": "batch_eval" if idx == 1 else "sweep_point", "weights": Ws, "biases": bs,
                "latents": Z, "queries": q}
    if idx == 2:
        Ws, bs = make_network(rng, L, H, bf16_weights=True)
        Z = make_latents(rng, 8, L)
        g = make_gbuffer(rng, 1920 if width is None else width, 1080 if height is None else height)
        return {"name": "frame_1080p_5lights", "weights": Ws, "biases": bs, "latents": Z, "gbuffer": g,
                "lights": lights_direct5()}
    if idx == 3:
        Ws, bs = make_network(rng, L, H, bf16_weights=True)
        Z = make_latents(rng, 8, L)
        g = make_gbuffer(rng, 3840 if width is None else width, 2160 if height is None else height)
        lights = lights_area16(rng)
        z_edit = rng.standard_normal(L).astype(np.float32)
        return {"name": "frame_4k_16lights_edit", "weights": Ws, "biases": bs, "latents": Z, "gbuffer": g,
                "lights": lights, "edit_material": 3, "edit_latent": z_edit}
    raise ValueError(idx)


# ---------------------------------------------------------------------------------------------------
# Inputs for the paper-structured decoder.  Data only, as above.
PD_LATENT = 64


def pd_layer_shapes(L=PD_LATENT, H=64, F=FEAT_DIM):
    """fusion (2 layers) + angular decoder (5 layers): [out, in] per layer."""
    return [(H, L + 24), (F, H), (H, F + 5), (H, H), (H, H), (H, H), (4, H)]


def make_pd_network(rng, L=PD_LATENT, H=64, F=FEAT_DIM, bf16_weights=True):
    """Xavier-uniform weights, biases 0.01*N(0,1).  The output biases are then shifted so that the synthetic network
    behaves like a BSDF: diffuse components around 1 (positive), log-mapped specular outputs around 3, i.e.
    S = (e^3 - 1)/100 ~ 0.2 for reflection.  Draw order: W1,b1,...,W7,b7."""
    Ws, bs = [], []
    for (n_out, n_in) in pd_layer_shapes(L, H, F):
        a = math.sqrt(6.0 / (n_in + n_out))
        W = rng.uniform(-a, a, size=(n_out, n_in)).astype(np.float32)
        b = (0.01 * rng.standard_normal(n_out)).astype(np.float32)
        Ws.append(round_to_bf16(W) if bf16_weights else W)
        bs.append(b)
    bs[6][0:2] += np.float32(1.0)
    bs[6][2:4] += np.float32(3.0)
    return Ws, bs


def make_albedos(rng, M):
    """[M][12] = kd_warp, kd_weft, ks_warp, ks_weft (RGB each) ~ U[0.05, 0.95)."""
    return rng.uniform(0.05, 0.95, size=(M, 12)).astype(np.float32)


def disk_direction(rng, n, transmit_fraction=0.0):
    """(x, y) uniform in the unit disk (Table 2 samples x, y in (-1,1) and keeps valid pairs),
    z = +sqrt(1 - x^2 - y^2), negated for a `transmit_fraction` of the samples (BTDF)."""
    r = np.sqrt(rng.random(n)) * 0.999
    phi = 2.0 * np.pi * rng.random(n)
    x, y = r * np.cos(phi), r * np.sin(phi)
    z = np.sqrt(np.maximum(0.0, 1.0 - x * x - y * y))
    if transmit_fraction > 0.0:
        z = np.where(rng.random(n) < transmit_fraction, -z, z)
    return np.stack([x, y, z], axis=1).astype(np.float32)


def make_pd_queries(rng, n, M):
    """Table 2: position U(0,1)^2, size U(0,1) or U(1,5) with equal probability, directions from
    the (x, y) disk; a quarter of the incoming directions lie below the surface (transmission).
    Draw order: u, v, size branch, size, wi, wo, material."""
    q = np.zeros(n, dtype=QUERY_DTYPE)
    q["u"] = rng.random(n).astype(np.float32)
    q["v"] = rng.random(n).astype(np.float32)
    big = rng.random(n) < 0.5
    s = rng.random(n)
    q["footprint"] = np.where(big, 1.0 + 4.0 * s, s).astype(np.float32)
    q["wi"] = disk_direction(rng, n, 0.25)
    q["wo"] = disk_direction(rng, n)
    q["material"] = rng.integers(0, M, n).astype(np.int32) if M > 1 else 0
    return q


def pd_config(kind, n=None, width=None, height=None, H=64, seed=None, M=8):
    """kind 'eval': batch of Table-2 queries; kind 'frame': the configs[2] G-buffer (footprint size = its uv
    derivative, in pattern units) with the five direct lights plus one point light BEHIND the fabric."""
    rng = np.random.default_rng({"eval": 11, "frame": 12}[kind] if seed is None else seed)
    Ws, bs = make_pd_network(rng, PD_LATENT, H)
    Z = make_latents(rng, M, PD_LATENT)
    A = make_albedos(rng, M)
    out = {"weights": Ws, "biases": bs, "latents": Z, "albedos": A}
    if kind == "eval":
        out["queries"] = make_pd_queries(rng, (1 << 20) if n is None else n, M)
    else:
        out["gbuffer"] = make_gbuffer(rng, 1920 if width is None else width, 1080 if height is None else height)
        back = np.zeros(1, dtype=LIGHT_DTYPE)
        back["type"] = 1
        back["vec"] = (0.2, -0.1, -0.6)
        back["rgb"] = (0.3, 0.35, 0.4)
        out["lights"] = np.concatenate([lights_direct5(), back])
    return out


# ---------------------------------------------------------------------------------------------------
# Inputs for the encoder tail.  Data only, as above.
def enc_layer_shapes(feat_width=256, hidden=128, latent=PD_LATENT):
    """in-projection, the two fully connected layers of the residual block, out-projection"""
    return [(hidden, feat_width + 2), (hidden, hidden), (hidden, hidden), (latent, hidden)]


def enc_config(feat_width=256, hidden=128, latent=PD_LATENT, seed=21, n_materials=8):
    """Xavier-uniform fp32 weights, biases 0.01*N(0,1); per material a stand-in for the ResNet-18 feature of its pattern
    textures (|N(0,1)|: post-ReLU, pooled features are non-negative) and appearance parameters roughness alpha ~ U(0.1, 0.9),
    height-field scaling beta ~ U(0.5, 2).  Draw order: E0,b0,...,E3,b3; features; alpha; beta."""
    rng = np.random.default_rng(seed)
    Ws, bs = [], []
    for (n_out, n_in) in enc_layer_shapes(feat_width, hidden, latent):
        a = math.sqrt(6.0 / (n_in + n_out))
        Ws.append(rng.uniform(-a, a, size=(n_out, n_in)).astype(np.float32))
        bs.append((0.01 * rng.standard_normal(n_out)).astype(np.float32))
    feats = np.abs(rng.standard_normal((n_materials, feat_width))).astype(np.float32)
    alpha = rng.uniform(0.1, 0.9, n_materials).astype(np.float32)
    beta = rng.uniform(0.5, 2.0, n_materials).astype(np.float32)
    return {"weights": Ws, "biases": bs, "features": feats, "alpha": alpha, "beta": beta}
