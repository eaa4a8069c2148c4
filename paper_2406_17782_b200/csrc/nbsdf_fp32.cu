// nbsdf_fp32.cu -- fp32 CUDA-core variant of the fused decoder (NBSDF_PREC_FP32): plain FMA, no TF32, no tensor
// cores.  A CTA owns a tile of 256 (H = 32) or 128 (H >= 64) queries; activations live in shared memory as
// [k][query] rows and every layer is a register-tiled product (4 x 8 outputs per thread at H = 64) with warp-uniform
// weight loads from L1.  Accumulation runs over k in index order, like the oracle's definition, in fp32.
// Decoder data flow: PAPER.md:164 (sec. 4.2 "Decoder"); per-frame recipe: PAPER.md:196.
#include "nbsdf_common.cuh"

namespace nbsdf {

struct Fp32Layout {
    uint32_t w_off[6];   // float offsets; layers 0..4 transposed Wt[k][N], layer 5 row-major W6[3][H]
    uint32_t b_off[6];
    uint32_t total;      // floats
};

__host__ __device__ inline Fp32Layout fp32_layout(int L, int H)
{
    Fp32Layout t;
    const int K[6] = { L + 3, H, H, kFeat + 6, H, H };
    const int N[6] = { H, H, kFeat, H, H, 3 };
    uint32_t off = 0;
    for (int l = 0; l < 6; ++l) {
        t.w_off[l] = off;
        off += (uint32_t)(K[l] * N[l]);
        off = (off + 3u) & ~3u;
        t.b_off[l] = off;
        off += (uint32_t)N[l];
        off = (off + 3u) & ~3u;
    }
    t.total = off;
    return t;
}

// Host-side packing used by nbsdf_create (declared in nbsdf_host.cu).
void pack_fp32(int L, int H, const nbsdf_weights* w, float* blob)
{
    Fp32Layout lay = fp32_layout(L, H);
    const int K[6] = { L + 3, H, H, kFeat + 6, H, H };
    const int N[6] = { H, H, kFeat, H, H, 3 };
    for (uint32_t i = 0; i < lay.total; ++i) blob[i] = 0.0f;
    for (int l = 0; l < 6; ++l) {
        for (int o = 0; o < N[l]; ++o) {
            for (int k = 0; k < K[l]; ++k) {
                float v = w->W[l][(size_t)o * K[l] + k];
                if (l < 5) blob[lay.w_off[l] + (size_t)k * N[l] + o] = v;
                else blob[lay.w_off[l] + (size_t)o * K[l] + k] = v;
            }
            blob[lay.b_off[l] + o] = w->b[l][o];
        }
    }
}

size_t fp32_blob_floats(int L, int H) { return fp32_layout(L, H).total; }

// ---------------------------------------------------------------------------------------------------------------------
// Register-tiled layers.  A CTA of 256 threads owns a tile of TQ * 32 queries (TQ = 8 for H = 32, 4 for H >= 64).
// Activations live in shared memory as [k][query] rows; lane l owns the TQ consecutive queries [TQ l, TQ l + TQ), warp w
// owns TN consecutive outputs, so that per k a thread reads TQ activations (LDS.128, conflict-free: a warp reads one
// contiguous row) and TN weights (warp-uniform LDG.128 that stay in L1) for TQ x TN FMAs -- 64 FMAs per 4 loads at
// H = 64 instead of the one shared-memory load per FMA-row of a thread-per-query layout.  Accumulation runs over k in
// index order in fp32 (plain FMA: no TF32, no tensor cores), like the oracle's definition.
constexpr int kThreads = 256;
constexpr int kWarps = kThreads / 32;

// out[n][q] = act(b[n] + sum_k Wt[k][n] in[k][q]) for n in [0, 8 TN), q in [0, 32 TQ); in/out: [.][32 TQ] floats
template <int TQ, int TN, bool kRelu>
__device__ __forceinline__ void dense_layer(const float* __restrict__ Wt, const float* __restrict__ b, int K,
                                            const float* in, float* out)
{
    constexpr int Q = 32 * TQ, N = kWarps * TN;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int q0 = lane * TQ, n0 = warp * TN;
    float acc[TN][TQ];
#pragma unroll
    for (int j = 0; j < TN; ++j) {
        const float bj = __ldg(b + n0 + j);
#pragma unroll
        for (int i = 0; i < TQ; ++i) acc[j][i] = bj;
    }
#pragma unroll 2
    for (int k = 0; k < K; ++k) {
        float a[TQ], w[TN];
#pragma unroll
        for (int i = 0; i < TQ; i += 4) {
            const float4 v = *reinterpret_cast<const float4*>(in + k * Q + q0 + i);
            a[i] = v.x; a[i + 1] = v.y; a[i + 2] = v.z; a[i + 3] = v.w;
        }
#pragma unroll
        for (int j = 0; j < TN; j += 4) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(Wt + (size_t)k * N + n0 + j));
            w[j] = v.x; w[j + 1] = v.y; w[j + 2] = v.z; w[j + 3] = v.w;
        }
#pragma unroll
        for (int j = 0; j < TN; ++j)
#pragma unroll
            for (int i = 0; i < TQ; ++i) acc[j][i] = fmaf(a[i], w[j], acc[j][i]);
    }
#pragma unroll
    for (int j = 0; j < TN; ++j)
#pragma unroll
        for (int i = 0; i < TQ; i += 4) {
            float4 v = make_float4(acc[j][i], acc[j][i + 1], acc[j][i + 2], acc[j][i + 3]);
            if (kRelu) { v.x = fmaxf(v.x, 0.0f); v.y = fmaxf(v.y, 0.0f); v.z = fmaxf(v.z, 0.0f); v.w = fmaxf(v.w, 0.0f); }
            *reinterpret_cast<float4*>(out + (n0 + j) * Q + q0 + i) = v;
        }
}

// MLP-A: x = [z, u', v', lf] in bufA -> feat in bufB rows [0, F)
template <int TQ, int TN>
__device__ __forceinline__ void mlp_a(const NetParams& net, const Fp32Layout& lay, float* bufA, float* bufB)
{
    const float* w = net.w32;
    dense_layer<TQ, TN, true>(w + lay.w_off[0], w + lay.b_off[0], net.L + 3, bufA, bufB);
    __syncthreads();
    dense_layer<TQ, TN, true>(w + lay.w_off[1], w + lay.b_off[1], net.H, bufB, bufA);
    __syncthreads();
    dense_layer<TQ, kFeat / kWarps, false>(w + lay.w_off[2], w + lay.b_off[2], net.H, bufA, bufB);
    __syncthreads();
}

// MLP-B: y = [feat, wi, wo] in bufB rows [0, F+6) -> rgb of query q (threads q < 32 TQ); bufB is preserved
template <int TQ, int TN>
__device__ __forceinline__ void mlp_b(const NetParams& net, const Fp32Layout& lay, float* bufA, float* bufB, float* bufC,
                                      float rgb[3])
{
    constexpr int Q = 32 * TQ;
    const float* w = net.w32;
    dense_layer<TQ, TN, true>(w + lay.w_off[3], w + lay.b_off[3], kFeat + 6, bufB, bufA);
    __syncthreads();
    dense_layer<TQ, TN, true>(w + lay.w_off[4], w + lay.b_off[4], net.H, bufA, bufC);
    __syncthreads();
    const int qi = threadIdx.x;
    if (qi < Q) {
        const float* W6 = w + lay.w_off[5];
        const float* b6 = w + lay.b_off[5];
        float o0 = 0.0f, o1 = 0.0f, o2 = 0.0f;
        for (int k = 0; k < net.H; ++k) {
            const float a = bufC[k * Q + qi];
            o0 = fmaf(a, __ldg(W6 + k), o0);
            o1 = fmaf(a, __ldg(W6 + net.H + k), o1);
            o2 = fmaf(a, __ldg(W6 + 2 * net.H + k), o2);
        }
        rgb[0] = softplus<false>(o0 + __ldg(b6 + 0));
        rgb[1] = softplus<false>(o1 + __ldg(b6 + 1));
        rgb[2] = softplus<false>(o2 + __ldg(b6 + 2));
    }
}

// shared memory: three activation buffers of Kmax x (32 TQ) floats
__host__ __device__ __forceinline__ int kmax_of(int L, int H)
{
    int k = H;
    if (L + 3 > k) k = L + 3;
    if (kFeat + 6 > k) k = kFeat + 6;
    return k;
}

template <int TQ, int TN>
__global__ void __launch_bounds__(kThreads) eval_fp32_kernel(NetParams net, const nbsdf_query* __restrict__ q,
                                                             const float* __restrict__ frames, int64_t n,
                                                             float* __restrict__ rgb_out)
{
    constexpr int Q = 32 * TQ;
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x;
    const int kmax = kmax_of(net.L, net.H);
    float* bufA = smem;
    float* bufB = bufA + kmax * Q;
    float* bufC = bufB + kmax * Q;
    const Fp32Layout lay = fp32_layout(net.L, net.H);

    // stages A1-A4: one query per thread (threads [0, Q)), straight into the [k][query] layout
    const int64_t i = (int64_t)blockIdx.x * Q + tid;
    const bool mine = tid < Q, live = mine && i < n;
    nbsdf_query rec;
    rec.u = rec.v = 0.0f; rec.footprint = 1.0f; rec.material = -1;
    rec.wi[0] = rec.wi[1] = 0.0f; rec.wi[2] = 1.0f;
    rec.wo[0] = rec.wo[1] = 0.0f; rec.wo[2] = 1.0f;
    if (live) rec = q[i];
    float wi[3] = { rec.wi[0], rec.wi[1], rec.wi[2] }, wo[3] = { rec.wo[0], rec.wo[1], rec.wo[2] };
    if (mine) {
        const int m = rec.material < 0 ? 0 : rec.material;
        if (frames != nullptr && live) {
            const float* f = frames + 6 * i;
            Frame fr = make_frame(f[0], f[1], f[2], f[3], f[4], f[5]);
            to_local(fr, rec.wi[0], rec.wi[1], rec.wi[2], wi);
            to_local(fr, rec.wo[0], rec.wo[1], rec.wo[2], wo);
        }
        for (int k = 0; k < net.L; ++k) bufA[k * Q + tid] = __ldg(net.latents + (size_t)m * net.L + k);
        bufA[(net.L + 0) * Q + tid] = wrap01(rec.u);
        bufA[(net.L + 1) * Q + tid] = wrap01(rec.v);
        bufA[(net.L + 2) * Q + tid] = log_footprint<false>(rec.footprint);
    }
    __syncthreads();
    mlp_a<TQ, TN>(net, lay, bufA, bufB);
    if (mine) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            bufB[(kFeat + c) * Q + tid] = wi[c];
            bufB[(kFeat + 3 + c) * Q + tid] = wo[c];
        }
    }
    __syncthreads();
    float rgb[3] = { 0.0f, 0.0f, 0.0f };
    mlp_b<TQ, TN>(net, lay, bufA, bufB, bufC, rgb);
    if (live) {
        const bool bg = rec.material < 0;
        rgb_out[3 * i + 0] = bg ? 0.0f : rgb[0];
        rgb_out[3 * i + 1] = bg ? 0.0f : rgb[1];
        rgb_out[3 * i + 2] = bg ? 0.0f : rgb[2];
    }
}

template <int TQ, int TN>
__global__ void __launch_bounds__(kThreads) shade_fp32_kernel(NetParams net, FrameParams fr, LightParams lights,
                                                              float* __restrict__ out)
{
    constexpr int Q = 32 * TQ;
    extern __shared__ __align__(16) float smem[];
    const int tid = threadIdx.x;
    const int kmax = kmax_of(net.L, net.H);
    float* bufA = smem;
    float* bufB = bufA + kmax * Q;
    float* bufC = bufB + kmax * Q;
    const Fp32Layout lay = fp32_layout(net.L, net.H);

    const int64_t p = (int64_t)blockIdx.x * Q + tid;
    const bool mine = tid < Q, live = mine && p < fr.n_pixels;
    float4 pos = make_float4(0.f, 0.f, 0.f, 1.f), nu = make_float4(0.f, 0.f, 1.f, 0.f), tv = make_float4(1.f, 0.f, 0.f, 0.f);
    int mat = -1;
    if (live) { pos = __ldg(fr.pos_fp + p); nu = __ldg(fr.nrm_u + p); tv = __ldg(fr.tan_v + p); mat = __ldg(fr.material + p); }
    const Frame f = make_frame(nu.x, nu.y, nu.z, tv.x, tv.y, tv.z);
    float wo[3];
    {
        const float vx = fr.cam[0] - pos.x, vy = fr.cam[1] - pos.y, vz = fr.cam[2] - pos.z;
        const float inv = rsqrtf(vx * vx + vy * vy + vz * vz);
        to_local(f, vx * inv, vy * inv, vz * inv, wo);
    }
    if (mine) {
        const int m = mat < 0 ? 0 : mat;
        for (int k = 0; k < net.L; ++k) bufA[k * Q + tid] = __ldg(net.latents + (size_t)m * net.L + k);
        bufA[(net.L + 0) * Q + tid] = wrap01(nu.w);
        bufA[(net.L + 1) * Q + tid] = wrap01(tv.w);
        bufA[(net.L + 2) * Q + tid] = log_footprint<false>(pos.w);
    }
    __syncthreads();
    mlp_a<TQ, TN>(net, lay, bufA, bufB);      // once per pixel (the spatial feature does not depend on wi/wo)
    if (mine) {
#pragma unroll
        for (int c = 0; c < 3; ++c) bufB[(kFeat + 3 + c) * Q + tid] = wo[c];
    }

    float acc[3] = { 0.0f, 0.0f, 0.0f };
    for (int l = 0; l < lights.n; ++l) {
        float wiw[3], E[3], wi[3], rgb[3] = { 0.0f, 0.0f, 0.0f };
        light_sample(lights.light[l], pos.x, pos.y, pos.z, wiw, E);
        to_local(f, wiw[0], wiw[1], wiw[2], wi);
        if (mine) {
#pragma unroll
            for (int c = 0; c < 3; ++c) bufB[(kFeat + c) * Q + tid] = wi[c];
        }
        __syncthreads();
        mlp_b<TQ, TN>(net, lay, bufA, bufB, bufC, rgb);
        const float cs = fmaxf(wi[2], 0.0f);
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[c] = fmaf(rgb[c] * E[c], cs, acc[c]);
        __syncthreads();                        // bufC / bufB's wi rows are rewritten by the next light
    }
    if (live) {
        const bool bg = mat < 0;
        out[3 * p + 0] = bg ? 0.0f : acc[0];
        out[3 * p + 1] = bg ? 0.0f : acc[1];
        out[3 * p + 2] = bg ? 0.0f : acc[2];
    }
}

template <int TQ>
static size_t fp32_smem(const NetParams& net) { return (size_t)3 * kmax_of(net.L, net.H) * 32 * TQ * sizeof(float); }

// H = 32: 8 queries x 4 outputs per thread; H = 64: 4 x 8 (128-query tiles: 96 KB, two CTAs per SM -- measured 16 % faster
// than 8 x 8 with one CTA per SM); H = 128: 4 x 16 (a 128-query tile keeps three buffers in 196 KB)
#define NBSDF_FP32_DISPATCH(CALL)                                  \
    switch (net.H) {                                               \
    case 32: { constexpr int TQ = 8, TN = 4; CALL; } break;        \
    case 64: { constexpr int TQ = 4, TN = 8; CALL; } break; \
    case 128: { constexpr int TQ = 4, TN = 16; CALL; } break;      \
    default: return cudaErrorInvalidValue;                         \
    }

cudaError_t init_fp32()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](const void* k) { if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024); };
    set((const void*)eval_fp32_kernel<8, 4>); set((const void*)eval_fp32_kernel<4, 8>); set((const void*)eval_fp32_kernel<4, 16>);
    set((const void*)shade_fp32_kernel<8, 4>); set((const void*)shade_fp32_kernel<4, 8>); set((const void*)shade_fp32_kernel<4, 16>);
    return e;
}

cudaError_t launch_eval_fp32(const NetParams& net, const nbsdf_query* q, const float* frames, int64_t n, float* rgb,
                             cudaStream_t s)
{
    NBSDF_FP32_DISPATCH((eval_fp32_kernel<TQ, TN><<<(unsigned)((n + 32 * TQ - 1) / (32 * TQ)), kThreads, fp32_smem<TQ>(net), s>>>(
        net, q, frames, n, rgb)))
    return cudaGetLastError();
}

cudaError_t launch_shade_fp32(const NetParams& net, const FrameParams& fr, const LightParams& lights, float* out,
                              cudaStream_t s)
{
    NBSDF_FP32_DISPATCH((shade_fp32_kernel<TQ, TN><<<(unsigned)((fr.n_pixels + 32 * TQ - 1) / (32 * TQ)), kThreads,
                                                   fp32_smem<TQ>(net), s>>>(net, fr, lights, out)))
    return cudaGetLastError();
}

// Latent interpolation: z_dst = (1 - t) z_a + t z_b, one thread per component, fp32.
__global__ void lerp_latents_kernel(float* __restrict__ latents, int L, int dst, int a, int b, float t)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < L) {
        const float za = latents[(size_t)a * L + i], zb = latents[(size_t)b * L + i];
        latents[(size_t)dst * L + i] = fmaf(t, zb, (1.0f - t) * za);
    }
}

cudaError_t launch_lerp_latents(float* latents, int L, int dst, int a, int b, float t, cudaStream_t s)
{
    lerp_latents_kernel<<<(L + 63) / 64, 64, 0, s>>>(latents, L, dst, a, b, t);
    return cudaGetLastError();
}

}  // namespace nbsdf
