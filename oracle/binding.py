"""Builds (gcc) and loads liboracle.so; argument marshalling only.  TEST INFRASTRUCTURE."""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nbsdf_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "nbsdf_oracle_paper.c"), os.path.join(_HERE, "nbsdf_oracle_encoder.c")]
_LIB = os.path.join(_HERE, "liboracle.so")

# wire format of the inputs (query = position, size, wi, wo + material latent id)
QUERY_DTYPE = np.dtype([("u", "<f4"), ("v", "<f4"), ("footprint", "<f4"), ("material", "<i4"),
                        ("wi", "<f4", (3,)), ("wo", "<f4", (3,))], align=False)
LIGHT_DTYPE = np.dtype([("type", "<i4"), ("vec", "<f4", (3,)), ("rgb", "<f4", (3,)),
                        ("emit_n", "<f4", (3,))], align=False)
assert QUERY_DTYPE.itemsize == 40 and LIGHT_DTYPE.itemsize == 40


class _Dims(C.Structure):
    _fields_ = [("latent_dim", C.c_int32), ("hidden", C.c_int32), ("feat_dim", C.c_int32),
                ("n_materials", C.c_int32)]


def build(force=False):
    """Compile the oracle with gcc (no fast-math, no contraction).  Building is not using."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-o", _LIB] + _SRCS + ["-lm"])
    return _LIB


_lib = None
_all_threads = 1


def _threads(n):
    """0 = all cores the process started with (an earlier 1-thread call must not stick)."""
    _load()
    return int(n) if n and n > 0 else _all_threads


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.oracle_softplus.restype = C.c_double
        lib.oracle_softplus.argtypes = [C.c_double]
        lib.oracle_wrap.restype = C.c_double
        lib.oracle_wrap.argtypes = [C.c_double]
        lib.oracle_log_footprint.restype = C.c_double
        lib.oracle_log_footprint.argtypes = [C.c_double]
        lib.oracle_to_local.restype = None
        lib.oracle_to_local.argtypes = [C.c_void_p] * 4
        lib.oracle_eval.restype = C.c_int
        lib.oracle_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                    C.c_int64, C.c_void_p, C.c_int]
        lib.oracle_shade_frame.restype = C.c_int
        lib.oracle_shade_frame.argtypes = [C.c_void_p] * 8 + [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p,
                                                              C.c_int, C.c_void_p, C.c_int]
        lib.oracle_max_threads.restype = C.c_int
        for name in ("oracle_leaky", "oracle_size01"):
            getattr(lib, name).restype = C.c_double
            getattr(lib, name).argtypes = [C.c_double]
        lib.oracle_inv_logmap.restype = C.c_double
        lib.oracle_inv_logmap.argtypes = [C.c_double, C.c_double]
        lib.oracle_oneblob.restype = None
        lib.oracle_oneblob.argtypes = [C.c_double, C.c_int, C.c_void_p]
        lib.oracle_lerp_latent.restype = None
        lib.oracle_lerp_latent.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p]
        lib.oracle_pd_eval.restype = C.c_int
        lib.oracle_pd_eval.argtypes = [C.c_void_p] * 7 + [C.c_int64, C.c_void_p, C.c_void_p, C.c_int]
        lib.oracle_pd_shade_frame.restype = C.c_int
        lib.oracle_pd_shade_frame.argtypes = [C.c_void_p] * 9 + [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p,
                                                                 C.c_int, C.c_void_p, C.c_int]
        lib.oracle_pd_shade_frame_px.restype = C.c_int
        lib.oracle_pd_shade_frame_px.argtypes = [C.c_void_p] * 10 + [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p,
                                                                     C.c_int, C.c_void_p, C.c_int]
        lib.oracle_encode_latent.restype = C.c_int
        lib.oracle_encode_latent.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p]
        global _all_threads
        _all_threads = int(lib.oracle_max_threads())      # before any call narrows the OpenMP team
        _lib = lib
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _pack_net(weights, biases, latents):
    """weights/biases: 6 arrays, W_k row-major [out][in]; latents [M][L].  Shapes define the dims."""
    Ws = [_f32(w) for w in weights]
    bs = [_f32(b).reshape(-1) for b in biases]
    Z = _f32(latents)
    assert len(Ws) == 6 and len(bs) == 6 and Z.ndim == 2
    M, L = Z.shape
    H, F = Ws[0].shape[0], Ws[2].shape[0]
    shapes = [(H, L + 3), (H, H), (F, H), (H, F + 6), (H, H), (3, H)]
    for w, b, s in zip(Ws, bs, shapes):
        assert w.shape == s and b.shape == (s[0],), (w.shape, b.shape, s)
    dims = _Dims(L, H, F, M)
    Wp = (C.c_void_p * 6)(*[w.ctypes.data for w in Ws])
    bp = (C.c_void_p * 6)(*[b.ctypes.data for b in bs])
    return dims, Wp, bp, Z, (Ws, bs)


def eval_queries(weights, biases, latents, queries, frames=None, n_threads=0):
    """fp64 decoder over a batch of QUERY_DTYPE records -> float64 [n][3]."""
    dims, Wp, bp, Z, _keep = _pack_net(weights, biases, latents)
    q = np.ascontiguousarray(queries, dtype=QUERY_DTYPE)
    n = q.shape[0]
    fr = None
    if frames is not None:
        fr = _f32(frames)
        assert fr.shape == (n, 6)
    mats = q["material"]
    assert n == 0 or int(mats.max()) < Z.shape[0], "material id out of range"
    out = np.empty((n, 3), dtype=np.float64)
    rc = _load().oracle_eval(C.byref(dims), Wp, bp, Z.ctypes.data, q.ctypes.data,
                             fr.ctypes.data if fr is not None else None, n, out.ctypes.data, _threads(n_threads))
    assert rc == 0
    return out


def shade_frame(weights, biases, latents, gbuffer, lights, first=0, count=None, n_threads=0):
    """fp64 frame shading.  gbuffer: dict(pos_fp, nrm_u, tan_v [h*w][4] f32, material [h*w] i32, cam_pos[3]).
    Returns float64 [count][3] for pixels [first, first+count)."""
    dims, Wp, bp, Z, _keep = _pack_net(weights, biases, latents)
    pos = _f32(gbuffer["pos_fp"]).reshape(-1, 4)
    nrm = _f32(gbuffer["nrm_u"]).reshape(-1, 4)
    tan = _f32(gbuffer["tan_v"]).reshape(-1, 4)
    mat = np.ascontiguousarray(gbuffer["material"], dtype=np.int32).reshape(-1)
    npx = mat.shape[0]
    assert pos.shape[0] == npx and nrm.shape[0] == npx and tan.shape[0] == npx
    cam = _f32(gbuffer["cam_pos"]).reshape(3)
    lt = np.ascontiguousarray(lights, dtype=LIGHT_DTYPE).reshape(-1)
    if count is None:
        count = npx - first
    assert 0 <= first and first + count <= npx
    assert npx == 0 or int(mat.max()) < Z.shape[0], "material id out of range"
    out = np.empty((count, 3), dtype=np.float64)
    rc = _load().oracle_shade_frame(C.byref(dims), Wp, bp, Z.ctypes.data, pos.ctypes.data, nrm.ctypes.data,
                                    tan.ctypes.data, mat.ctypes.data, first, count, cam.ctypes.data,
                                    lt.ctypes.data if lt.shape[0] else None, lt.shape[0], out.ctypes.data,
                                    _threads(n_threads))
    assert rc == 0
    return out


def softplus(x):
    return _load().oracle_softplus(float(x))


def wrap(x):
    return _load().oracle_wrap(float(x))


def log_footprint(x):
    return _load().oracle_log_footprint(float(x))


def to_local(n, t, w):
    n = np.ascontiguousarray(n, dtype=np.float64)
    t = np.ascontiguousarray(t, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    out = np.empty(3, dtype=np.float64)
    _load().oracle_to_local(n.ctypes.data, t.ctypes.data, w.ctypes.data, out.ctypes.data)
    return out


def max_threads():
    _load()
    return _all_threads


# ---------------------------------------------------------------------------------------------------
# paper-structured decoder (nbsdf_oracle_paper.c)
def _pack_pd(weights, biases, latents, albedos):
    """weights/biases: 7 arrays (fusion 2 + angular decoder 5), W_k row-major [out][in]; latents [M][L];
    albedos [M][12] = kd_warp, kd_weft, ks_warp, ks_weft (RGB each)."""
    Ws = [_f32(w) for w in weights]
    bs = [_f32(b).reshape(-1) for b in biases]
    Z = _f32(latents)
    A = _f32(albedos)
    assert len(Ws) == 7 and len(bs) == 7 and Z.ndim == 2
    M, L = Z.shape
    assert A.shape == (M, 12)
    H, F = Ws[0].shape[0], Ws[1].shape[0]
    shapes = [(H, L + 24), (F, H), (H, F + 5), (H, H), (H, H), (H, H), (4, H)]
    for w, b, s in zip(Ws, bs, shapes):
        assert w.shape == s and b.shape == (s[0],), (w.shape, b.shape, s)
    dims = _Dims(L, H, F, M)
    Wp = (C.c_void_p * 7)(*[w.ctypes.data for w in Ws])
    bp = (C.c_void_p * 7)(*[b.ctypes.data for b in bs])
    return dims, Wp, bp, Z, A, (Ws, bs)


def pd_eval_queries(weights, biases, latents, albedos, queries, frames=None, n_threads=0, components=False):
    """fp64 paper-structured decoder over QUERY_DTYPE records (footprint = size in pattern units; wo.z unused)
    -> float64 [n][3] (and [n][4] = C_warp, C_weft, S_warp, S_weft when components=True)."""
    dims, Wp, bp, Z, A, _keep = _pack_pd(weights, biases, latents, albedos)
    q = np.ascontiguousarray(queries, dtype=QUERY_DTYPE)
    n = q.shape[0]
    fr = None
    if frames is not None:
        fr = _f32(frames)
        assert fr.shape == (n, 6)
    assert n == 0 or int(q["material"].max()) < Z.shape[0], "material id out of range"
    out = np.empty((n, 3), dtype=np.float64)
    comp = np.empty((n, 4), dtype=np.float64) if components else None
    rc = _load().oracle_pd_eval(C.byref(dims), Wp, bp, Z.ctypes.data, A.ctypes.data, q.ctypes.data,
                                fr.ctypes.data if fr is not None else None, n, out.ctypes.data,
                                comp.ctypes.data if components else None, _threads(n_threads))
    assert rc == 0
    return (out, comp) if components else out


def pd_shade_frame(weights, biases, latents, albedos, gbuffer, lights, first=0, count=None, n_threads=0):
    """fp64 frame shading with the paper-structured decoder (|cos| weighting; pos_fp.w = footprint size).
    gbuffer may carry "albedo": a per-pixel plane [h*w][12] that replaces the material's table row."""
    dims, Wp, bp, Z, A, _keep = _pack_pd(weights, biases, latents, albedos)
    pos = _f32(gbuffer["pos_fp"]).reshape(-1, 4)
    nrm = _f32(gbuffer["nrm_u"]).reshape(-1, 4)
    tan = _f32(gbuffer["tan_v"]).reshape(-1, 4)
    mat = np.ascontiguousarray(gbuffer["material"], dtype=np.int32).reshape(-1)
    npx = mat.shape[0]
    cam = _f32(gbuffer["cam_pos"]).reshape(3)
    lt = np.ascontiguousarray(lights, dtype=LIGHT_DTYPE).reshape(-1)
    if count is None:
        count = npx - first
    assert 0 <= first and first + count <= npx
    assert npx == 0 or int(mat.max()) < Z.shape[0], "material id out of range"
    out = np.empty((count, 3), dtype=np.float64)
    apx = None
    if gbuffer.get("albedo") is not None:
        apx = _f32(gbuffer["albedo"]).reshape(-1, 12)
        assert apx.shape[0] == npx
    rc = _load().oracle_pd_shade_frame_px(C.byref(dims), Wp, bp, Z.ctypes.data, A.ctypes.data,
                                          apx.ctypes.data if apx is not None else None, pos.ctypes.data,
                                          nrm.ctypes.data, tan.ctypes.data, mat.ctypes.data, first, count,
                                          cam.ctypes.data, lt.ctypes.data if lt.shape[0] else None, lt.shape[0],
                                          out.ctypes.data, _threads(n_threads))
    assert rc == 0
    return out


def oneblob(s, k=8):
    out = np.empty(k, dtype=np.float64)
    _load().oracle_oneblob(float(s), int(k), out.ctypes.data)
    return out


def leaky(x):
    return _load().oracle_leaky(float(x))


def size01(x):
    return _load().oracle_size01(float(x))


def inv_logmap(y, k):
    return _load().oracle_inv_logmap(float(y), float(k))


def lerp_latent(za, zb, t):
    za, zb = _f32(za).reshape(-1), _f32(zb).reshape(-1)
    assert za.shape == zb.shape
    out = np.empty(za.shape[0], dtype=np.float64)
    _load().oracle_lerp_latent(za.ctypes.data, zb.ctypes.data, za.shape[0], float(t), out.ctypes.data)
    return out


class _EncDims(C.Structure):
    _fields_ = [("feat_width", C.c_int32), ("hidden", C.c_int32), ("latent_dim", C.c_int32)]


def encode_latent(weights, biases, feature, alpha, beta):
    """fp64 encoder tail (nbsdf_oracle_encoder.c): weights/biases = 4 arrays E0 [He][Fr+2], E1, E2 [He][He], E3 [L][He];
    feature [Fr] fp32; returns z float64 [L]."""
    Ws = [_f32(w) for w in weights]
    bs = [_f32(b).reshape(-1) for b in biases]
    f = _f32(feature).reshape(-1)
    He, L, Fr = Ws[0].shape[0], Ws[3].shape[0], f.shape[0]
    for w, b, s in zip(Ws, bs, [(He, Fr + 2), (He, He), (He, He), (L, He)]):
        assert w.shape == s and b.shape == (s[0],), (w.shape, b.shape, s)
    dims = _EncDims(Fr, He, L)
    Wp = (C.c_void_p * 4)(*[w.ctypes.data for w in Ws])
    bp = (C.c_void_p * 4)(*[b.ctypes.data for b in bs])
    out = np.empty(L, dtype=np.float64)
    rc = _load().oracle_encode_latent(C.byref(dims), Wp, bp, f.ctypes.data, float(alpha), float(beta), out.ctypes.data)
    assert rc == 0
    return out
