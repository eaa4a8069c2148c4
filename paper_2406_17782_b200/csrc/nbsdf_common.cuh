// nbsdf_common.cuh -- shared declarations of the CUDA library (host context + kernel parameter blocks)
// and the per-query input assembly (stages A2-A4, C1 of DESIGN.md).  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nbsdf.h"

namespace nbsdf {

constexpr int kFeat = 32;          // F: feature width of MLP-A (BASELINE.json configs[0])
constexpr int kTileRows = 128;     // queries per tile = TMEM lanes = threads per warpgroup

// Device pointers + dims handed to every kernel (by value).
struct NetParams {
    const float* latents;   // [M][L] fp32 latent table ("material latent vector")
    const float* w32;       // fp32 path: transposed, padded weights + biases (see pack_fp32)
    const uint8_t* wimg_eval;    // tensor path: shared-memory image for nbsdf_eval (5 layers, feature layer merged)
    const uint8_t* wimg_shade;   // tensor path: shared-memory image for nbsdf_shade_frame (6 layers)
    const float* albedos;        // paper-structured decoder: [M][12] fp32 (kd_warp, kd_weft, ks_warp, ks_weft) x RGB
    int32_t L, H, M;
};

struct LightParams {
    nbsdf_light light[NBSDF_MAX_LIGHTS];   // directional vec already normalised on the host
    int32_t n;
};

// What an EVAL launch passes in place of the 1.3-KB light table it never reads (kernel parameters are copied at every
// launch: at 2^12..2^16 queries the launch is latency-bound and the parameter block is part of that latency).
struct NoLightParams {
    nbsdf_light light[1];
    int32_t n;
};

struct FrameParams {
    const float4* pos_fp;
    const float4* nrm_u;
    const float4* tan_v;
    const int32_t* material;
    const float4* albedo;        // paper-structured contexts: per-pixel [12] albedos (3 float4 per pixel), or NULL
    int64_t n_pixels;
    float cam[3];
};

// ---------------------------------------------------------------------------------------------
// Stage A2: wrap to the pattern period (period 1).  floor-based, so negatives land in [0,1].
__device__ __forceinline__ float wrap01(float x) { return x - floorf(x); }

// Stage A3: log2 of the footprint clamped to [2^-20, 2^4].  fmaxf/fminf also turn fp <= 0 (and NaN) into the bound.
template <bool kFast>
__device__ __forceinline__ float log_footprint(float fp)
{
    float c = fminf(fmaxf(fp, 9.5367431640625e-07f), 16.0f);
    return kFast ? __log2f(c) : log2f(c);
}

struct Frame {
    float t[3], b[3], n[3];
};

// Stage A4: orthonormal frame from (n, tangent hint): n^ = n/|n|, t' = t - n^(n^.t), degenerate t' replaced by
// e_k - n^ n^_k with k = argmin |n^_k| (lowest k on ties), b^ = n^ x t^.
__device__ __forceinline__ Frame make_frame(float nx, float ny, float nz, float tx, float ty, float tz)
{
    Frame f;
    float inv = rsqrtf(nx * nx + ny * ny + nz * nz);
    nx *= inv; ny *= inv; nz *= inv;
    float nt = nx * tx + ny * ty + nz * tz;
    tx -= nx * nt; ty -= ny * nt; tz -= nz * nt;
    float tt = tx * tx + ty * ty + tz * tz;
    if (tt < 1e-12f) {
        float ax = fabsf(nx), ay = fabsf(ny), az = fabsf(nz);
        int k = 0;
        float am = ax;
        if (ay < am) { k = 1; am = ay; }
        if (az < am) { k = 2; }
        float nk = k == 0 ? nx : (k == 1 ? ny : nz);
        tx = (k == 0 ? 1.0f : 0.0f) - nx * nk;
        ty = (k == 1 ? 1.0f : 0.0f) - ny * nk;
        tz = (k == 2 ? 1.0f : 0.0f) - nz * nk;
        tt = tx * tx + ty * ty + tz * tz;
    }
    inv = rsqrtf(tt);
    tx *= inv; ty *= inv; tz *= inv;
    f.n[0] = nx; f.n[1] = ny; f.n[2] = nz;
    f.t[0] = tx; f.t[1] = ty; f.t[2] = tz;
    f.b[0] = ny * tz - nz * ty;
    f.b[1] = nz * tx - nx * tz;
    f.b[2] = nx * ty - ny * tx;
    return f;
}

__device__ __forceinline__ void to_local(const Frame& f, float x, float y, float z, float out[3])
{
    out[0] = x * f.t[0] + y * f.t[1] + z * f.t[2];
    out[1] = x * f.b[0] + y * f.b[1] + z * f.b[2];
    out[2] = x * f.n[0] + y * f.n[1] + z * f.n[2];
}

// Stage C1: direction to light l and its irradiance factor E at world position x.
__device__ __forceinline__ void light_sample(const nbsdf_light& lt, float px, float py, float pz, float wi[3], float E[3])
{
    if (lt.type == 0) {
        wi[0] = lt.vec[0]; wi[1] = lt.vec[1]; wi[2] = lt.vec[2];
        E[0] = lt.rgb[0]; E[1] = lt.rgb[1]; E[2] = lt.rgb[2];
    } else {
        float vx = lt.vec[0] - px, vy = lt.vec[1] - py, vz = lt.vec[2] - pz;
        float d2 = vx * vx + vy * vy + vz * vz;
        float inv = rsqrtf(d2);
        wi[0] = vx * inv; wi[1] = vy * inv; wi[2] = vz * inv;
        float fac = 1.0f;
        if (lt.emit_n[0] != 0.0f || lt.emit_n[1] != 0.0f || lt.emit_n[2] != 0.0f)
            fac = fmaxf(0.0f, -(wi[0] * lt.emit_n[0] + wi[1] * lt.emit_n[1] + wi[2] * lt.emit_n[2]));
        float s = fac * inv * inv;
        E[0] = lt.rgb[0] * s; E[1] = lt.rgb[1] * s; E[2] = lt.rgb[2] * s;
    }
}

// Stage B7: softplus(x) = ln(1 + e^x), beta = 1, no threshold.
template <bool kFast>
__device__ __forceinline__ float softplus(float x)
{
    if (kFast) {
        float t = __expf(-fabsf(x));
        // log1p(t): series below 0.01 keeps the tail (x << 0) relatively accurate, MUFU.LG2 above
        float l = t < 0.01f ? t * (1.0f - t * (0.5f - t * 0.33333334f)) : __logf(1.0f + t);
        return fmaxf(x, 0.0f) + l;
    }
    return x > 0.0f ? x + log1pf(expf(-x)) : log1pf(expf(x));
}

// ---------------------------------------------------------------------------------------------
// launchers implemented in nbsdf_fp32.cu / nbsdf_tc.cu; return the cudaError_t of the launch
cudaError_t launch_eval_fp32(const NetParams& net, const nbsdf_query* q, const float* frames, int64_t n, float* rgb,
                             cudaStream_t s);
cudaError_t launch_shade_fp32(const NetParams& net, const FrameParams& fr, const LightParams& lights, float* out,
                              cudaStream_t s);
cudaError_t launch_eval_tc(const NetParams& net, int precision, int num_sms, const nbsdf_query* q, const float* frames,
                           int64_t n, float* rgb, cudaStream_t s);
cudaError_t launch_shade_tc(const NetParams& net, int precision, int num_sms, const FrameParams& fr,
                            const LightParams& lights, float* out, cudaStream_t s);
cudaError_t init_tc(int L, int H);       // cudaFuncSetAttribute for the instantiations in use
cudaError_t init_fp32();

// shared-memory image layout of the tensor path, computed identically on host (packing) and device (carving).
// Biases are folded into the contractions: every layer's input vector is extended by kBiasCols constant entries
// (c0, c1, c2) and the weight rows by (b0/c0, b1/c1, b2/c2), where b0 + b1 + b2 is the 16-bit three-way split of
// the fp32 bias -- the tensor core then adds the bias in its fp32 accumulator at full precision and the epilogue
// is left with ReLU + pack only.  Layers 1 and 4 take the constants inside their K padding; the K = H layers get
// one extra 16-wide K step whose A operand is a per-warpgroup constant TMEM block.
constexpr int kBiasCols = 3;

// constant fed in bias input column j: fp16 scales the residual parts up out of the subnormal range
__host__ __device__ constexpr float tc_bias_const(bool bf16, int j)
{
    return bf16 ? 1.0f : (j == 0 ? 1.0f : (j == 1 ? 0.000244140625f /* 2^-12 */ : 0.00006103515625f /* 2^-14 */));
}

struct TcLayout {
    int n_layers;            // 6, or 5 when the linear feature layer is merged into layer 4 (eval image)
    int K1p, K4p;            // padded K of layers 1 and 4 (multiples of 16), bias columns included
    int Kp[6];               // padded K of every layer as issued (K = H layers: H + 16)
    int Kbias[6];            // input index of the first bias column of every layer
    uint32_t w_off[6];       // byte offset of each layer's weight tiles (1024-aligned)
    uint32_t w_rows[6];      // padded N (rows) of each layer
    uint32_t total;          // bytes of the image (multiple of 16)
};

__host__ __device__ constexpr int pad16(int k) { return (k + 15) & ~15; }

// merged == false: the six layers as defined (nbsdf_shade_frame, where the feature is reused across lights; and H = 128).
// merged == true : nbsdf_eval's image for H <= 64.  The feature layer is linear, so
//                  W4[:, :F] (W3 h2 + b3) + W4[:, F:] [wi, wo] + b4 == (W4f W3) h2 + W4a [wi, wo] + (W4f b3 + b4):
//                  layers 3 and 4 become ONE H x (H + 6) layer, one MMA round and one epilogue fewer per tile.
//                  Multiply-adds: H (H + 6) merged vs 2 F H + 6 H separate -- equal at H = 64 (F = 32), fewer at H = 32,
//                  twice as many at H = 128 (which is why H = 128 keeps six layers).  Its last K step reads
//                  [wi, wo, c0, c1, c2] from a per-warpgroup tail block instead of the CTA-wide bias-constant block.
#ifndef NBSDF_EVAL_MERGE_MAX_H
#define NBSDF_EVAL_MERGE_MAX_H 64
#endif
__host__ __device__ constexpr bool tc_eval_merged(int H) { return H <= NBSDF_EVAL_MERGE_MAX_H; }

__host__ __device__ constexpr TcLayout tc_layout(int L, int H, bool merged)
{
    TcLayout t{};
    t.K1p = pad16(L + 3 + kBiasCols);
    t.K4p = pad16(kFeat + 6 + kBiasCols);
    t.n_layers = merged ? 5 : 6;
    const int K6[6] = { t.K1p, H + 16, H + 16, t.K4p, H + 16, H + 16 };
    const int Kb6[6] = { L + 3, H, H, kFeat + 6, H, H };
    const int N6[6] = { H, H, kFeat, H, H, 16 };
    const int K5[6] = { t.K1p, H + 16, H + 16, H + 16, H + 16, 0 };
    const int Kb5[6] = { L + 3, H, H + 6, H, H, 0 };
    const int N5[6] = { H, H, H, H, 16, 0 };
    uint32_t off = 0;
    for (int l = 0; l < t.n_layers; ++l) {
        const int K = merged ? K5[l] : K6[l];
        const int N = merged ? N5[l] : N6[l];
        t.Kp[l] = K;
        t.Kbias[l] = merged ? Kb5[l] : Kb6[l];
        t.w_off[l] = off;
        t.w_rows[l] = (uint32_t)N;
        off += (uint32_t)((K + 63) / 64) * (uint32_t)N * 128u;   // N rows x 128 B per 64-wide K block
    }
    t.total = (off + 15u) & ~15u;
    return t;
}

// ---------------------------------------------------------------------------------------------
// Paper-structured decoder (nbsdf_tc_paper.cu): seven layers, same image format as above.
//   1: [z(64), blob(24), c] -> H     2: H -> F       (fusion)
//   3: [feat(F), wi(3), wo(2), c] -> H   4: H -> H   5: H -> H (+ skip, added in the epilogue)   6: H -> H   7: H -> 4
constexpr int kPdLatent = 64;
constexpr int kPdBlob = 24;
constexpr int kPdLayers = 7;
constexpr float kPdSlope = 0.01f;

struct PdLayout {
    int Kp[kPdLayers];            // padded K as issued
    int Kbias[kPdLayers];         // input index of the first bias column
    uint32_t w_off[kPdLayers];
    uint32_t w_rows[kPdLayers];   // padded N
    uint32_t total;
};

__host__ __device__ constexpr PdLayout pd_layout(int H)
{
    PdLayout t{};
    const int K[kPdLayers] = { pad16(kPdLatent + kPdBlob + kBiasCols), H + 16, pad16(kFeat + 5 + kBiasCols), H + 16, H + 16, H + 16, H + 16 };
    const int Kb[kPdLayers] = { kPdLatent + kPdBlob, H, kFeat + 5, H, H, H, H };
    const int N[kPdLayers] = { H, kFeat, H, H, H, H, 16 };
    uint32_t off = 0;
    for (int l = 0; l < kPdLayers; ++l) {
        t.Kp[l] = K[l];
        t.Kbias[l] = Kb[l];
        t.w_off[l] = off;
        t.w_rows[l] = (uint32_t)N[l];
        off += (uint32_t)((K[l] + 63) / 64) * (uint32_t)N[l] * 128u;
    }
    t.total = (off + 15u) & ~15u;
    return t;
}

cudaError_t launch_lerp_latents(float* latents, int L, int dst, int a, int b, float t, cudaStream_t s);   // nbsdf_fp32.cu
cudaError_t init_pd(int H);
cudaError_t launch_eval_pd(const NetParams& net, int num_sms, const nbsdf_query* q, const float* frames, int64_t n, float* rgb,
                           cudaStream_t s);
cudaError_t launch_shade_pd(const NetParams& net, int num_sms, const FrameParams& fr, const LightParams& lights, float* out,
                            cudaStream_t s);

}  // namespace nbsdf
