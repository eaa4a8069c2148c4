"""ctypes binding of libnbsdf.so -- same call names as include/nbsdf.h, argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; PyTorch supplies device memory and the
stream.  There is no fallback: if the library cannot be built/loaded, or the device is not sm_100, the calls raise.
"""
import ctypes as C

import numpy as np

from . import buildlib
from .synth import LIGHT_DTYPE, QUERY_DTYPE  # wire formats (numpy dtypes), no arithmetic

NBSDF_OK, NBSDF_E_INVALID, NBSDF_E_UNSUPPORTED, NBSDF_E_CUDA, NBSDF_E_NOMEM = 0, -1, -2, -3, -4
NBSDF_PREC_FP32, NBSDF_PREC_BF16, NBSDF_PREC_FP16 = 0, 1, 2
PRECISIONS = {"fp32": NBSDF_PREC_FP32, "bf16": NBSDF_PREC_BF16, "fp16": NBSDF_PREC_FP16}
NBSDF_MAX_LIGHTS = 32
EXPORTS = ["nbsdf_create", "nbsdf_set_latents", "nbsdf_eval", "nbsdf_shade_frame", "nbsdf_destroy",
           "nbsdf_last_error", "nbsdf_launch_count", "nbsdf_create_paper", "nbsdf_set_albedos", "nbsdf_lerp_latents",
           "nbsdf_set_encoder", "nbsdf_encode_latent", "nbsdf_encode_latent_static", "nbsdf_get_latents"]


class NbsdfError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"nbsdf status {status}: {msg}")
        self.status = status


class _Config(C.Structure):
    _fields_ = [("latent_dim", C.c_int32), ("hidden", C.c_int32), ("feat_dim", C.c_int32),
                ("max_materials", C.c_int32), ("precision", C.c_int32), ("device", C.c_int32)]


class _Weights(C.Structure):
    _fields_ = [("W", C.c_void_p * 6), ("b", C.c_void_p * 6)]


class _PaperWeights(C.Structure):
    _fields_ = [("W", C.c_void_p * 7), ("b", C.c_void_p * 7)]


class _EncoderWeights(C.Structure):
    _fields_ = [("W", C.c_void_p * 4), ("b", C.c_void_p * 4), ("feat_width", C.c_int32), ("hidden", C.c_int32)]


class _GBuffer(C.Structure):
    _fields_ = [("pos_fp", C.c_void_p), ("nrm_u", C.c_void_p), ("tan_v", C.c_void_p), ("material", C.c_void_p),
                ("width", C.c_int32), ("height", C.c_int32), ("cam_pos", C.c_float * 3), ("albedo", C.c_void_p)]


_lib = None


def load():
    """Build (if stale) and dlopen libnbsdf.so; declare the prototypes of include/nbsdf.h."""
    global _lib
    if _lib is None:
        lib = C.CDLL(buildlib.build())
        lib.nbsdf_create.restype = C.c_int
        lib.nbsdf_create.argtypes = [C.POINTER(_Config), C.POINTER(_Weights), C.POINTER(C.c_void_p)]
        lib.nbsdf_set_latents.restype = C.c_int
        lib.nbsdf_set_latents.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        lib.nbsdf_eval.restype = C.c_int
        lib.nbsdf_eval.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        lib.nbsdf_shade_frame.restype = C.c_int
        lib.nbsdf_shade_frame.argtypes = [C.c_void_p, C.POINTER(_GBuffer), C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        lib.nbsdf_destroy.restype = None
        lib.nbsdf_destroy.argtypes = [C.c_void_p]
        lib.nbsdf_last_error.restype = C.c_char_p
        lib.nbsdf_last_error.argtypes = [C.c_void_p]
        lib.nbsdf_launch_count.restype = C.c_int64
        lib.nbsdf_launch_count.argtypes = [C.c_void_p]
        lib.nbsdf_create_paper.restype = C.c_int
        lib.nbsdf_create_paper.argtypes = [C.POINTER(_Config), C.POINTER(_PaperWeights), C.POINTER(C.c_void_p)]
        lib.nbsdf_lerp_latents.restype = C.c_int
        lib.nbsdf_lerp_latents.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float, C.c_void_p]
        lib.nbsdf_set_albedos.restype = C.c_int
        lib.nbsdf_set_albedos.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        lib.nbsdf_set_encoder.restype = C.c_int
        lib.nbsdf_set_encoder.argtypes = [C.c_void_p, C.POINTER(_EncoderWeights)]
        lib.nbsdf_encode_latent.restype = C.c_int
        lib.nbsdf_encode_latent.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_float, C.c_float, C.c_void_p]
        lib.nbsdf_encode_latent_static.restype = C.c_int
        lib.nbsdf_encode_latent_static.argtypes = [C.c_int32, C.POINTER(_EncoderWeights), C.c_int32, C.c_void_p, C.c_float,
                                                   C.c_float, C.c_void_p, C.c_void_p]
        lib.nbsdf_get_latents.restype = C.c_int
        lib.nbsdf_get_latents.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        _lib = lib
    return _lib


def _check(rc, ctx):
    if rc != NBSDF_OK:
        raise NbsdfError(rc, load().nbsdf_last_error(ctx).decode())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream))


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def nbsdf_create(weights, biases, latent_dim, hidden, max_materials, precision="fp16", device=0, feat_dim=32):
    """weights/biases: 6 host arrays, W_k row-major [out][in] fp32.  Returns the opaque context handle."""
    Ws = [np.ascontiguousarray(w, dtype=np.float32) for w in weights]
    bs = [np.ascontiguousarray(b, dtype=np.float32).reshape(-1) for b in biases]
    L, H, F = latent_dim, hidden, feat_dim
    for w, b, s in zip(Ws, bs, [(H, L + 3), (H, H), (F, H), (H, F + 6), (H, H), (3, H)]):
        if w.shape != s or b.shape != (s[0],):
            raise ValueError(f"layer shape {w.shape}/{b.shape}, expected {s}")
    cfg = _Config(L, H, F, max_materials, PRECISIONS.get(precision, precision), device)
    wt = _Weights((C.c_void_p * 6)(*[w.ctypes.data for w in Ws]), (C.c_void_p * 6)(*[b.ctypes.data for b in bs]))
    ctx = C.c_void_p()
    rc = load().nbsdf_create(C.byref(cfg), C.byref(wt), C.byref(ctx))
    _check(rc, None)
    return ctx


def nbsdf_create_paper(weights, biases, hidden, max_materials, precision="fp16", device=0, latent_dim=64, feat_dim=32):
    """Paper-structured decoder (include/nbsdf.h): 7 host arrays each, W_k row-major [out][in] fp32."""
    Ws = [np.ascontiguousarray(w, dtype=np.float32) for w in weights]
    bs = [np.ascontiguousarray(b, dtype=np.float32).reshape(-1) for b in biases]
    L, H, F = latent_dim, hidden, feat_dim
    for w, b, s in zip(Ws, bs, [(H, L + 24), (F, H), (H, F + 5), (H, H), (H, H), (H, H), (4, H)]):
        if w.shape != s or b.shape != (s[0],):
            raise ValueError(f"layer shape {w.shape}/{b.shape}, expected {s}")
    cfg = _Config(L, H, F, max_materials, PRECISIONS.get(precision, precision), device)
    wt = _PaperWeights((C.c_void_p * 7)(*[w.ctypes.data for w in Ws]), (C.c_void_p * 7)(*[b.ctypes.data for b in bs]))
    ctx = C.c_void_p()
    rc = load().nbsdf_create_paper(C.byref(cfg), C.byref(wt), C.byref(ctx))
    _check(rc, None)
    return ctx


def nbsdf_set_albedos(ctx, first, albedos_host, stream=None):
    a = np.ascontiguousarray(albedos_host, dtype=np.float32)
    a = a.reshape(1, -1) if a.ndim == 1 else a
    if a.shape[1] != 12:
        raise ValueError("albedos: 12 values per material (kd_warp, kd_weft, ks_warp, ks_weft) x RGB")
    _check(load().nbsdf_set_albedos(ctx, first, a.shape[0], a.ctypes.data, _stream(stream)), ctx)


def nbsdf_set_latents(ctx, first, latents_host, stream=None):
    z = np.ascontiguousarray(latents_host, dtype=np.float32)
    z = z.reshape(1, -1) if z.ndim == 1 else z
    _check(load().nbsdf_set_latents(ctx, first, z.shape[0], z.ctypes.data, _stream(stream)), ctx)


def nbsdf_set_encoder(ctx, weights, biases):
    """Encoder tail (include/nbsdf.h): 4 host arrays each, E0 [He][Fr+2], E1, E2 [He][He], E3 [L][He], fp32."""
    Ws = [np.ascontiguousarray(w, dtype=np.float32) for w in weights]
    bs = [np.ascontiguousarray(b, dtype=np.float32).reshape(-1) for b in biases]
    if len(Ws) != 4 or len(bs) != 4:
        raise ValueError("encoder tail: 4 layers")
    He, Fr, L = Ws[0].shape[0], Ws[0].shape[1] - 2, Ws[3].shape[0]
    for w, b, s in zip(Ws, bs, [(He, Fr + 2), (He, He), (He, He), (L, He)]):
        if w.shape != s or b.shape != (s[0],):
            raise ValueError(f"layer shape {w.shape}/{b.shape}, expected {s}")
    ew = _EncoderWeights((C.c_void_p * 4)(*[w.ctypes.data for w in Ws]), (C.c_void_p * 4)(*[b.ctypes.data for b in bs]), Fr, He)
    _check(load().nbsdf_set_encoder(ctx, C.byref(ew)), ctx)


def nbsdf_encode_latent(ctx, row, feature_host, alpha, beta, stream=None):
    f = np.ascontiguousarray(feature_host, dtype=np.float32).reshape(-1)
    _check(load().nbsdf_encode_latent(ctx, int(row), f.ctypes.data if f.size else None, float(alpha), float(beta),
                                      _stream(stream)), ctx)


def nbsdf_encode_latent_static(weights_dev, biases_dev, feature_dev, alpha, beta, z_dev, device=0, stream=None):
    """The encoder tail without any allocation (include/nbsdf.h): for callers that cannot cudaMalloc.  weights_dev /
    biases_dev: 4 contiguous CUDA float32 tensors each, E0 [He][Fr+2], E1, E2 [He][He], E3 [L][He], read in place;
    feature_dev: CUDA float32 [Fr] (None when Fr == 0); z_dev: CUDA float32 [L], receives the latent.  Shapes are only
    read off the tensors here; the size limits (He <= 256, Fr <= 1022, L <= 64) are the library's to enforce."""
    if len(weights_dev) != 4 or len(biases_dev) != 4:
        raise ValueError("encoder tail: 4 layers")
    He, Fr, L = weights_dev[0].shape[0], weights_dev[0].shape[1] - 2, weights_dev[3].shape[0]
    for w, b, s in zip(weights_dev, biases_dev, [(He, Fr + 2), (He, He), (He, He), (L, He)]):
        if tuple(w.shape) != s or b.numel() != s[0] or not (w.is_cuda and b.is_cuda and w.is_contiguous() and b.is_contiguous()):
            raise ValueError(f"layer {tuple(w.shape)}/{tuple(b.shape)}: expected contiguous CUDA tensors of shape {s}")
    if z_dev.numel() != L or (Fr and (feature_dev is None or feature_dev.numel() != Fr)):
        raise ValueError("feature must hold Fr floats and z_dev L floats")
    ew = _EncoderWeights((C.c_void_p * 4)(*[w.data_ptr() for w in weights_dev]),
                         (C.c_void_p * 4)(*[b.data_ptr() for b in biases_dev]), Fr, He)
    _check(load().nbsdf_encode_latent_static(int(device), C.byref(ew), L, _ptr(feature_dev) if Fr else None, float(alpha),
                                             float(beta), _ptr(z_dev), _stream(stream)), None)


def nbsdf_get_latents(ctx, first, count, latent_dim, stream=None):
    """Rows [first, first+count) of the context's latent table as a host float32 array [count][latent_dim] (blocks)."""
    out = np.empty((count, latent_dim), dtype=np.float32)
    _check(load().nbsdf_get_latents(ctx, int(first), int(count), out.ctypes.data, _stream(stream)), ctx)
    return out


def nbsdf_lerp_latents(ctx, dst, a, b, t, stream=None):
    _check(load().nbsdf_lerp_latents(ctx, int(dst), int(a), int(b), float(t), _stream(stream)), ctx)


def nbsdf_eval(ctx, q_dev, frames_dev, n, rgb_dev, stream=None):
    """q_dev: CUDA tensor holding n 40-byte records; frames_dev: CUDA float32 [n][6] or None; rgb_dev: CUDA float32 [n][3]."""
    _check(load().nbsdf_eval(ctx, _ptr(q_dev), _ptr(frames_dev), n, _ptr(rgb_dev), _stream(stream)), ctx)


def nbsdf_shade_frame(ctx, gbuf, lights_host, radiance_dev, stream=None):
    """gbuf: dict(pos_fp, nrm_u, tan_v: CUDA float32 [h*w][4]; material: CUDA int32 [h*w]; width; height; cam_pos)."""
    g = _GBuffer(gbuf["pos_fp"].data_ptr(), gbuf["nrm_u"].data_ptr(), gbuf["tan_v"].data_ptr(),
                 gbuf["material"].data_ptr(), int(gbuf["width"]), int(gbuf["height"]),
                 (C.c_float * 3)(*[float(c) for c in gbuf["cam_pos"]]),
                 gbuf["albedo"].data_ptr() if gbuf.get("albedo") is not None else None)
    lt = np.ascontiguousarray(lights_host, dtype=LIGHT_DTYPE).reshape(-1)
    _check(load().nbsdf_shade_frame(ctx, C.byref(g), lt.ctypes.data if lt.shape[0] else None, lt.shape[0],
                                    _ptr(radiance_dev), _stream(stream)), ctx)


def nbsdf_destroy(ctx):
    load().nbsdf_destroy(ctx)


def nbsdf_launch_count(ctx):
    return int(load().nbsdf_launch_count(ctx))


# ---- small conveniences for tests / bench: numpy <-> device tensors (plumbing only) ----
def queries_to_device(q, device="cuda"):
    import torch
    q = np.ascontiguousarray(q, dtype=QUERY_DTYPE)
    return torch.from_numpy(q.view(np.uint8).reshape(-1).copy()).to(device)


def gbuffer_to_device(g, device="cuda"):
    import torch
    out = {k: torch.from_numpy(np.ascontiguousarray(g[k])).to(device) for k in ("pos_fp", "nrm_u", "tan_v", "material")}
    if g.get("albedo") is not None:
        out["albedo"] = torch.from_numpy(np.ascontiguousarray(g["albedo"], dtype=np.float32)).to(device)
    out.update(width=g["width"], height=g["height"], cam_pos=[float(c) for c in g["cam_pos"]])
    return out
