/*
 * nbsdf.h -- C ABI of libnbsdf.so: the B200 (sm_100a) neural woven-fabric BSDF decoder.
 *
 * The calls follow the problem statement of "Real-time Neural Woven Fabric Rendering"
 * (arXiv 2406.17782; citations are /root/reference/PAPER.md line numbers):
 *   decoder signature (z, position, size, wi, wo) -> BSDF value ......... PAPER.md:160, Eq. 7 at 149
 *   two-MLP decoder (spatial fusion MLP-A, angular decoder MLP-B) ....... PAPER.md:164 (sec. 4.2 "Decoder")
 *   per-frame recipe (query + lighting -> decoder -> BSDF x lighting) ... PAPER.md:196 (sec. 4.3 "Rendering")
 *   editing = replace the material latent vector between frames ......... PAPER.md:198 (sec. 4.3 "Editing")
 * The network shapes are those of BASELINE.json configs (DESIGN.md "Readings" #1):
 *   MLP-A: [z(L), u', v', log2 fp] -> H (ReLU) -> H (ReLU) -> F (linear feature), F = 32
 *   MLP-B: [feat(F), wi(3), wo(3)] -> H (ReLU) -> H (ReLU) -> 3, softplus
 *
 * Conventions
 *   - All pointers are plain C pointers; each parameter says whether it is HOST or DEVICE memory.
 *   - The caller owns every query / G-buffer / output buffer and the CUDA stream (passed as void* =
 *     cudaStream_t; NULL = the legacy default stream).  The library owns only its packed weights,
 *     latent table and light staging, all released by nbsdf_destroy.  HOST arrays handed to
 *     nbsdf_create / nbsdf_set_latents / nbsdf_shade_frame(lights) are copied before the call returns.
 *   - nbsdf_eval / nbsdf_shade_frame / nbsdf_set_latents / nbsdf_set_albedos / nbsdf_lerp_latents only enqueue work
 *     on the given stream and return.  The one exception: host rows handed to nbsdf_set_latents / nbsdf_set_albedos /
 *     nbsdf_encode_latent are staged in a ring of 8 pinned slots, and a 9th edit issued while the 1st is still
 *     outstanding BLOCKS THE HOST until the stream has reached the 1st edit -- the copy is stream-ordered, so that means
 *     until every kernel queued ahead of it has finished.  Up to 8 outstanding edits never block.
 *   - A context is NOT thread-safe: its staging ring, launch counter and error text are plain members.  Use one context
 *     per host thread, or serialise the calls on a context yourself.  Different contexts are independent.
 *   - CUDA graphs: nbsdf_eval / nbsdf_shade_frame / nbsdf_lerp_latents may be captured.  nbsdf_set_latents /
 *     nbsdf_set_albedos / nbsdf_encode_latent return NBSDF_E_INVALID on a capturing stream and enqueue nothing (a replay
 *     would re-read a pinned slot the host has reused): issue edits between replays.
 *   - Work is ordered by the stream: a set_latents is visible to every later launch on the same stream
 *     (the editing guarantee of PAPER.md:198).  Every call works on cfg.device and restores the caller's current
 *     CUDA device before it returns.
 *   - Every call returns an nbsdf_status and never throws or aborts; nbsdf_last_error gives text.
 *     On NBSDF_E_INVALID nothing is launched.  There is no CPU fallback: a device that is not
 *     sm_100 makes nbsdf_create fail with NBSDF_E_UNSUPPORTED.
 *   - Directions are unit length; wi points from the surface to the light, wo to the viewer.  Without a
 *     frame they are already local (+z = macro normal).  material in [0, max_materials); a negative
 *     material yields exactly (0,0,0); material >= max_materials is undefined behaviour.
 *     Inputs must be finite; a non-finite input yields an unspecified (finite or NaN) value for THAT row only and
 *     never a fault.
 *   - Operand precision: NBSDF_PREC_FP16 (the default of the Python binding) meets max 1e-2 / mean 2e-3 against the
 *     fp64 definition on every supported dims with ~8x margin.  NBSDF_PREC_BF16 exists for networks whose activations
 *     exceed the fp16 range; its 8-bit significands cannot hold the max bound for hidden = 32 (any latent_dim) or for
 *     (latent_dim 32, hidden 64) (0.5e-2 .. 1.2e-2), and nbsdf_create REJECTS bf16 there with
 *     NBSDF_E_UNSUPPORTED rather than serve it at a looser tolerance; at the remaining dims the five-seed emulation stays <= 0.8e-2.
 */
#ifndef NBSDF_H
#define NBSDF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nbsdf_ctx nbsdf_ctx; /* opaque, owned by the library */

typedef enum {
    NBSDF_OK = 0,
    NBSDF_E_INVALID = -1,     /* NULL pointer, negative size, misaligned buffer, range error */
    NBSDF_E_UNSUPPORTED = -2, /* device is not sm_100, or dims outside the supported set */
    NBSDF_E_CUDA = -3,        /* a CUDA runtime call failed; see nbsdf_last_error */
    NBSDF_E_NOMEM = -4
} nbsdf_status;

typedef enum {
    NBSDF_PREC_FP32 = 0, /* CUDA-core variant: fp32 FMA everywhere (no TF32, no tensor cores); <= 1e-5 vs oracle */
    NBSDF_PREC_BF16 = 1, /* tcgen05 tensor cores, bf16 operands, fp32 accumulate in TMEM */
    NBSDF_PREC_FP16 = 2  /* tcgen05 tensor cores, fp16 operands (bf16-stored weights convert exactly), fp32 accumulate */
} nbsdf_precision;

/* Supported: latent_dim in {8,16,32}, hidden in {32,64,128}, feat_dim == 32, 1 <= max_materials <= 64. */
typedef struct {
    int32_t latent_dim;    /* L */
    int32_t hidden;        /* H */
    int32_t feat_dim;      /* F */
    int32_t max_materials; /* M: rows of the latent table */
    int32_t precision;     /* nbsdf_precision */
    int32_t device;        /* CUDA device ordinal */
} nbsdf_config;

/* HOST pointers, fp32, row-major W[k][out][in], y = W x + b.  Layer input widths:
 * W[0]: H x (L+3), W[1]: H x H, W[2]: F x H, W[3]: H x (F+6), W[4]: H x H, W[5]: 3 x H.
 * In the tensor-core precisions the weights are rounded to the operand type (RNE) at create; biases,
 * latents, queries and outputs stay fp32. */
typedef struct {
    const float* W[6];
    const float* b[6];
} nbsdf_weights;

/* One shading query, 40 bytes, array-of-structs (position, size, wi, wo + material). */
typedef struct {
    float u, v;       /* footprint position in pattern units; wrapped to [0,1) by the library */
    float footprint;  /* footprint side length in pattern units; log2 of clamp(., 2^-20, 2^4) is fed to MLP-A */
    int32_t material; /* row of the latent table; < 0 => output (0,0,0) */
    float wi[3];      /* to the light */
    float wo[3];      /* to the viewer */
} nbsdf_query;

/* Headless G-buffer, DEVICE planes, 52 bytes per pixel (+ 48 with an albedo plane); pixel index = y * width + x. */
typedef struct {
    const float* pos_fp;     /* [h*w][4]: world x, y, z, footprint   (16-byte aligned) */
    const float* nrm_u;      /* [h*w][4]: shading normal nx, ny, nz, u               */
    const float* tan_v;      /* [h*w][4]: tangent hint tx, ty, tz, v                 */
    const int32_t* material; /* [h*w]; < 0 = background => radiance (0,0,0)          */
    int32_t width, height;
    float cam_pos[3];        /* pinhole position; wo = normalize(cam_pos - x)        */
    const float* albedo;     /* NULL, or (contexts made by nbsdf_create_paper only) [h*w][12]: per-pixel kd_warp, kd_weft,
                              * ks_warp, ks_weft (RGB each) that replace the material's row of the albedo table in Eq. 8 --
                              * "spatial-varying appearances when applying albedo maps, by computing k_d and k_s via
                              * mipmapping"; the mip-mapped texture fetch is the renderer's, its result is
                              * this plane.  16-byte aligned.  Non-NULL on an nbsdf_create context => NBSDF_E_INVALID. */
} nbsdf_gbuffer;

/* type 0: directional, vec = direction TO the light (normalised by the library), rgb = radiance E.
 * type 1: point, vec = position, rgb = intensity I;  E = I * max(0, -wi . emit_n) / |vec - x|^2,
 *         emit_n = (0,0,0) => isotropic (factor 1). */
typedef struct {
    int32_t type;
    float vec[3];
    float rgb[3];
    float emit_n[3];
} nbsdf_light;

#define NBSDF_MAX_LIGHTS 32

/* Builds a decoder context on cfg->device: validates dims, packs the weights for the chosen precision
 * (tensor-core paths: operand type, K padded to 16, 128-byte-swizzled K-major tiles as tcgen05 reads them),
 * allocates the latent table (zero-filled).  weights: HOST, copied.  *out receives the context. */
int nbsdf_create(const nbsdf_config* cfg, const nbsdf_weights* weights, nbsdf_ctx** out);

/* Overwrites rows [first, first+count) of the material latent table ("update the material
 * latent vector").  latents_host: HOST, count x L fp32, copied before return; the device update is enqueued
 * on cuda_stream and ordered before later launches on it.  first+count > max_materials => NBSDF_E_INVALID. */
int nbsdf_set_latents(nbsdf_ctx* ctx, int32_t first, int32_t count, const float* latents_host, void* cuda_stream);

/* Latent interpolation / extrapolation on the device (sec. 6.3 "Interpolation"): row dst of the latent
 * table becomes (1 - t) * row a + t * row b, in fp32, by a small kernel enqueued on cuda_stream (ordered like
 * nbsdf_set_latents; no host round trip).  t may lie outside [0, 1] (extrapolation); dst may equal a or b.
 * Rows outside [0, max_materials) => NBSDF_E_INVALID. */
int nbsdf_lerp_latents(nbsdf_ctx* ctx, int32_t dst, int32_t a, int32_t b, float t, void* cuda_stream);

/* ---- Encoder tail on the device (sec. 4.2 "Encoder", 168 Fig. 3 caption; editing path PAPER.md:198) ----
 * The fully connected residual block that turns a pre-computed ResNet feature of the fabric pattern plus the appearance
 * parameters (roughness alpha, height-field scaling beta) into a material latent vector (DESIGN.md sec. 12 for the
 * readings): x = [feature(Fr), alpha, beta];
 *   e0 = lrelu(W[0] x + b[0]);  r = lrelu(W[1] e0 + b[1]);  e2 = lrelu(W[2] r + b[2] + e0);  z = W[3] e2 + b[3]
 * with leaky-ReLU slope 0.01, all in fp32.  HOST pointers, fp32, row-major [out][in]:
 * W[0]: He x (Fr+2), W[1], W[2]: He x He, W[3]: L x He with L = the context's latent_dim.
 * Supported: hidden He in {32, 64, 128, 256}, 0 <= feat_width Fr <= 1022; else NBSDF_E_UNSUPPORTED. */
typedef struct {
    const float* W[4];
    const float* b[4];
    int32_t feat_width; /* Fr */
    int32_t hidden;     /* He: 128 in the paper */
} nbsdf_encoder_weights;

/* Installs (or replaces) the encoder tail of a context: weights are copied to the device before the call returns
 * (a set-up call: it synchronises with the device).  Works on contexts made by nbsdf_create or nbsdf_create_paper. */
int nbsdf_set_encoder(nbsdf_ctx* ctx, const nbsdf_encoder_weights* weights);

/* Runs the encoder tail for one material and writes the result into row `row` of the latent table: one small kernel
 * enqueued on cuda_stream, ordered like nbsdf_set_latents (visible to every later launch on the stream; no host round
 * trip, no synchronisation).  feature_host: HOST, Fr fp32, copied before return.  NBSDF_E_INVALID if no encoder has
 * been installed or row is out of range. */
int nbsdf_encode_latent(nbsdf_ctx* ctx, int32_t row, const float* feature_host, float alpha, float beta, void* cuda_stream);

/* The encoder tail for callers that cannot allocate device memory -- a renderer whose own pool already holds the whole
 * GPU, or a frame loop that cannot take the device-wide synchronisation cudaMalloc / cudaFree imply.  (The two calls
 * above allocate: weight blob, staging slots, pinned ring.)  This call allocates NOTHING, on the device or the host, and
 * needs no context: same arithmetic as nbsdf_encode_latent (fp32, leaky-ReLU slope 0.01), run as one small kernel per
 * layer (4 launches) enqueued on cuda_stream of `device`; the caller's current device is restored on return.
 *   weights_dev: HOST struct whose W[] / b[] are DEVICE pointers, fp32, row-major [out][in], shapes as listed above
 *                with L = latent_dim; read in place (no packed copy), so they must stay valid until the work has run.
 *   feature_dev: DEVICE, Fr fp32 (may be NULL when Fr == 0).   z_dev: DEVICE, latent_dim fp32, receives z -- e.g. the
 *                caller's own latent buffer; to put it into a context's table copy it to the host for nbsdf_set_latents.
 * Scratch: the activations between the launches live in ONE fixed 3-KB array inside the library image (a static
 * __device__ array: every GPU that loads the library holds it until the process exits).  Hence
 *   - limits: hidden <= 256 (any value, not only the four above), feat_width <= 1022, latent_dim <= 64; beyond them
 *     the call returns NBSDF_E_UNSUPPORTED and launches nothing;
 *   - every call on a GPU shares the array.  Calls on one stream are ordered and safe; calls that can overlap on the
 *     GPU (two streams with no event between them, two threads) race on it and give wrong latents.  Nothing in it needs
 *     clearing between calls: each launch reads only what an earlier launch of the same call wrote;
 *   - the FIRST call on each device also looks up the array's device address (cudaGetSymbolAddress) and caches it:
 *     make that call during set-up, before any stream capture.
 * Errors: as everywhere; the text is at nbsdf_last_error(NULL). */
int nbsdf_encode_latent_static(int32_t device, const nbsdf_encoder_weights* weights_dev, int32_t latent_dim,
                               const float* feature_dev, float alpha, float beta, float* z_dev, void* cuda_stream);

/* Reads rows [first, first+count) of the latent table back: latents_host: HOST, count x L fp32.  Enqueued on cuda_stream
 * after the edits already queued there; BLOCKS until that copy has finished (a debugging / checking call, not part of
 * the frame loop).  Rows out of range => NBSDF_E_INVALID. */
int nbsdf_get_latents(nbsdf_ctx* ctx, int32_t first, int32_t count, float* latents_host, void* cuda_stream);

/* Batched decoder inference: stages A1-A4, B1-B7 of DESIGN.md in one fused kernel.
 * q_dev: DEVICE, n records, 16-byte aligned.  frames_dev: DEVICE [n][6] = (normal, tangent hint) per query in
 * the space of wi/wo, or NULL when wi/wo are already local.  rgb_dev: DEVICE [n][3] fp32, 16-byte aligned.
 * n == 0 is a no-op returning NBSDF_OK; n >= 2^37 per call is NBSDF_E_INVALID (tile indices are 32-bit and
 * the kernels look three rounds of tiles ahead). */
int nbsdf_eval(nbsdf_ctx* ctx, const nbsdf_query* q_dev, const float* frames_dev, int64_t n, float* rgb_dev,
               void* cuda_stream);

/* Frame shading: per pixel, MLP-A once, MLP-B once per light,
 * radiance[p] = sum_l rgb(z_m, uv, fp, wi_l, wo) * E_l * max(0, wi_l,local.z), lights in index order.
 * gbuf: HOST struct holding DEVICE plane pointers.  lights_host: HOST, n_lights <= NBSDF_MAX_LIGHTS, copied.
 * radiance_dev: DEVICE [h][w][3] fp32, 16-byte aligned.  width * height >= 2^37 => NBSDF_E_INVALID. */
int nbsdf_shade_frame(nbsdf_ctx* ctx, const nbsdf_gbuffer* gbuf, const nbsdf_light* lights_host, int32_t n_lights,
                      float* radiance_dev, void* cuda_stream);

/* ---- Decoder with the paper's own structure ----
 * latent 64; one-blob encoding of (u', v', size/5) with 8 bins each, 3 -> 24 channels;
 * fusion:          W[0]: H x (64+24) leaky ReLU,  W[1]: F x H leaky ReLU                   ("two fully connected layers")
 * angular decoder: W[2]: H x (F+5) on [feat, wi.xyz, wo.xy],  W[3]: H x H,  W[4]: H x H + skip from W[2]'s output,
 *                  W[5]: H x H,  W[6]: 4 x H (linear); leaky ReLU (slope 0.01) after all but the last
 *                  ("five fully connected layers with one skip connection").
 * Outputs (C_warp, C_weft, g(S_warp), g(S_weft)), g(x) = ln(k x + 1), k = 100 when wi_local.z >= 0 and 1000 below
 * (PAPER.md:172-177); the library inverts g and combines with the material's albedos (Eq. 8):
 *   rgb = kd_warp C_warp + kd_weft C_weft + ks_warp S_warp + ks_weft S_weft.
 * HOST pointers, fp32, row-major [out][in], copied.  Supported: latent_dim 64, hidden 64, feat_dim 32,
 * precision NBSDF_PREC_FP16 (tensor cores); anything else => NBSDF_E_UNSUPPORTED (bf16 operands cannot meet the
 * tolerance through the log-mapped specular outputs and are rejected rather than served).
 * A context made here is used with the same nbsdf_set_latents / nbsdf_eval / nbsdf_shade_frame calls:
 *   nbsdf_query.footprint and pos_fp.w then hold the footprint SIZE in multiples of the pattern size (clamped to
 *   [0, 5]), wo.z is ignored, and nbsdf_shade_frame weights each light by |wi_local.z| (transmission contributes). */
typedef struct {
    const float* W[7];
    const float* b[7];
} nbsdf_paper_weights;

int nbsdf_create_paper(const nbsdf_config* cfg, const nbsdf_paper_weights* weights, nbsdf_ctx** out);

/* Overwrites rows [first, first+count) of the albedo table of a paper-structured context: 12 fp32 per material,
 * kd_warp, kd_weft, ks_warp, ks_weft (RGB each); the table starts zero-filled.  PAPER.md:198: "to edit albedos ... no
 * encoder inference is needed".  albedos_host: HOST, copied before return; ordered on cuda_stream like set_latents.
 * NBSDF_E_INVALID on a context made by nbsdf_create. */
int nbsdf_set_albedos(nbsdf_ctx* ctx, int32_t first, int32_t count, const float* albedos_host, void* cuda_stream);

/* Frees everything the context owns.  The caller must have synchronised the streams it used.  NULL is allowed. */
void nbsdf_destroy(nbsdf_ctx* ctx);

/* Text of the last error on this context (or of the last failed nbsdf_create when ctx == NULL).  Never NULL. */
const char* nbsdf_last_error(const nbsdf_ctx* ctx);

/* Number of kernel launches this context has enqueued so far (bench.py's gpu_launches). */
int64_t nbsdf_launch_count(const nbsdf_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* NBSDF_H */
