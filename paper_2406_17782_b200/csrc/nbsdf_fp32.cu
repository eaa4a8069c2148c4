// nbsdf_fp32.cu -- fp32 CUDA-core variant of the fused decoder (NBSDF_PREC_FP32): plain FMA, no TF32, no tensor
// cores.  One thread per query; activations live in shared memory as [k][thread] columns (conflict-free), each
// layer is computed in register chunks of 32 outputs with warp-uniform (broadcast) weight loads from L1.
// Accumulation runs over k in index order, like the oracle's definition, in fp32.
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

constexpr int kThreads = 128;

// out[n][tid] = act(b[n] + sum_k Wt[k][n] * in[k][tid]) for n in [0, N), N % 32 == 0
template <bool kRelu>
__device__ __forceinline__ void dense_layer(const float* __restrict__ Wt, const float* __restrict__ b, int K, int N,
                                            const float* in, float* out, int tid)
{
    for (int n0 = 0; n0 < N; n0 += 32) {
        float acc[32];
#pragma unroll
        for (int j = 0; j < 32; j += 4) {
            float4 bv = __ldg(reinterpret_cast<const float4*>(b + n0 + j));
            acc[j] = bv.x; acc[j + 1] = bv.y; acc[j + 2] = bv.z; acc[j + 3] = bv.w;
        }
        for (int k = 0; k < K; ++k) {
            const float a = in[k * kThreads + tid];
            const float4* wr = reinterpret_cast<const float4*>(Wt + (size_t)k * N + n0);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                float4 wv = __ldg(wr + j);
                acc[4 * j + 0] = fmaf(a, wv.x, acc[4 * j + 0]);
                acc[4 * j + 1] = fmaf(a, wv.y, acc[4 * j + 1]);
                acc[4 * j + 2] = fmaf(a, wv.z, acc[4 * j + 2]);
                acc[4 * j + 3] = fmaf(a, wv.w, acc[4 * j + 3]);
            }
        }
#pragma unroll
        for (int j = 0; j < 32; ++j) out[(n0 + j) * kThreads + tid] = kRelu ? fmaxf(acc[j], 0.0f) : acc[j];
    }
}

// MLP-A: x = [z, u', v', lf] in bufA -> feat in bufB rows [0, F)
__device__ __forceinline__ void mlp_a(const NetParams& net, const Fp32Layout& lay, float* bufA, float* bufB, int tid)
{
    const float* w = net.w32;
    dense_layer<true>(w + lay.w_off[0], w + lay.b_off[0], net.L + 3, net.H, bufA, bufB, tid);
    dense_layer<true>(w + lay.w_off[1], w + lay.b_off[1], net.H, net.H, bufB, bufA, tid);
    dense_layer<false>(w + lay.w_off[2], w + lay.b_off[2], net.H, kFeat, bufA, bufB, tid);
}

// MLP-B: y = [feat, wi, wo] in bufB rows [0, F+6) -> rgb (softplus); bufB is preserved (feat reused across lights)
__device__ __forceinline__ void mlp_b(const NetParams& net, const Fp32Layout& lay, float* bufA, float* bufB, float* bufC,
                                      int tid, float rgb[3])
{
    const float* w = net.w32;
    dense_layer<true>(w + lay.w_off[3], w + lay.b_off[3], kFeat + 6, net.H, bufB, bufA, tid);
    dense_layer<true>(w + lay.w_off[4], w + lay.b_off[4], net.H, net.H, bufA, bufC, tid);
    const float* W6 = w + lay.w_off[5];
    const float* b6 = w + lay.b_off[5];
    float o0 = 0.0f, o1 = 0.0f, o2 = 0.0f;
    for (int k = 0; k < net.H; ++k) {
        const float a = bufC[k * kThreads + tid];
        o0 = fmaf(a, __ldg(W6 + k), o0);
        o1 = fmaf(a, __ldg(W6 + net.H + k), o1);
        o2 = fmaf(a, __ldg(W6 + 2 * net.H + k), o2);
    }
    rgb[0] = softplus<false>(o0 + __ldg(b6 + 0));
    rgb[1] = softplus<false>(o1 + __ldg(b6 + 1));
    rgb[2] = softplus<false>(o2 + __ldg(b6 + 2));
}

// shared memory: three activation buffers of Kmax x 128 floats
__device__ __forceinline__ int kmax_of(const NetParams& net)
{
    int k = net.H;
    if (net.L + 3 > k) k = net.L + 3;
    if (kFeat + 6 > k) k = kFeat + 6;
    return k;
}

__global__ void __launch_bounds__(kThreads) eval_fp32_kernel(NetParams net, const nbsdf_query* __restrict__ q,
                                                             const float* __restrict__ frames, int64_t n,
                                                             float* __restrict__ rgb_out)
{
    extern __shared__ float smem[];
    const int tid = threadIdx.x;
    const int kmax = kmax_of(net);
    float* bufA = smem;
    float* bufB = bufA + kmax * kThreads;
    float* bufC = bufB + kmax * kThreads;
    const Fp32Layout lay = fp32_layout(net.L, net.H);

    const int64_t i = (int64_t)blockIdx.x * kThreads + tid;
    const bool live = i < n;
    nbsdf_query rec;
    rec.u = rec.v = 0.0f; rec.footprint = 1.0f; rec.material = -1;
    rec.wi[0] = rec.wi[1] = 0.0f; rec.wi[2] = 1.0f;
    rec.wo[0] = rec.wo[1] = 0.0f; rec.wo[2] = 1.0f;
    if (live) rec = q[i];
    const int m = rec.material < 0 ? 0 : rec.material;
    float wi[3] = { rec.wi[0], rec.wi[1], rec.wi[2] }, wo[3] = { rec.wo[0], rec.wo[1], rec.wo[2] };
    if (frames != nullptr && live) {
        const float* f = frames + 6 * i;
        Frame fr = make_frame(f[0], f[1], f[2], f[3], f[4], f[5]);
        to_local(fr, rec.wi[0], rec.wi[1], rec.wi[2], wi);
        to_local(fr, rec.wo[0], rec.wo[1], rec.wo[2], wo);
    }
    for (int k = 0; k < net.L; ++k) bufA[k * kThreads + tid] = __ldg(net.latents + (size_t)m * net.L + k);
    bufA[(net.L + 0) * kThreads + tid] = wrap01(rec.u);
    bufA[(net.L + 1) * kThreads + tid] = wrap01(rec.v);
    bufA[(net.L + 2) * kThreads + tid] = log_footprint<false>(rec.footprint);
    mlp_a(net, lay, bufA, bufB, tid);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        bufB[(kFeat + c) * kThreads + tid] = wi[c];
        bufB[(kFeat + 3 + c) * kThreads + tid] = wo[c];
    }
    float rgb[3];
    mlp_b(net, lay, bufA, bufB, bufC, tid, rgb);
    if (live) {
        const bool bg = rec.material < 0;
        rgb_out[3 * i + 0] = bg ? 0.0f : rgb[0];
        rgb_out[3 * i + 1] = bg ? 0.0f : rgb[1];
        rgb_out[3 * i + 2] = bg ? 0.0f : rgb[2];
    }
}

__global__ void __launch_bounds__(kThreads) shade_fp32_kernel(NetParams net, FrameParams fr, LightParams lights,
                                                              float* __restrict__ out)
{
    extern __shared__ float smem[];
    const int tid = threadIdx.x;
    const int kmax = kmax_of(net);
    float* bufA = smem;
    float* bufB = bufA + kmax * kThreads;
    float* bufC = bufB + kmax * kThreads;
    const Fp32Layout lay = fp32_layout(net.L, net.H);

    const int64_t p = (int64_t)blockIdx.x * kThreads + tid;
    const bool live = p < fr.n_pixels;
    float4 pos = make_float4(0.f, 0.f, 0.f, 1.f), nu = make_float4(0.f, 0.f, 1.f, 0.f), tv = make_float4(1.f, 0.f, 0.f, 0.f);
    int mat = -1;
    if (live) { pos = __ldg(fr.pos_fp + p); nu = __ldg(fr.nrm_u + p); tv = __ldg(fr.tan_v + p); mat = __ldg(fr.material + p); }
    const int m = mat < 0 ? 0 : mat;
    const Frame f = make_frame(nu.x, nu.y, nu.z, tv.x, tv.y, tv.z);
    float vx = fr.cam[0] - pos.x, vy = fr.cam[1] - pos.y, vz = fr.cam[2] - pos.z;
    float inv = rsqrtf(vx * vx + vy * vy + vz * vz);
    float wo[3];
    to_local(f, vx * inv, vy * inv, vz * inv, wo);

    for (int k = 0; k < net.L; ++k) bufA[k * kThreads + tid] = __ldg(net.latents + (size_t)m * net.L + k);
    bufA[(net.L + 0) * kThreads + tid] = wrap01(nu.w);
    bufA[(net.L + 1) * kThreads + tid] = wrap01(tv.w);
    bufA[(net.L + 2) * kThreads + tid] = log_footprint<false>(pos.w);
    mlp_a(net, lay, bufA, bufB, tid);      // once per pixel (the spatial feature does not depend on wi/wo)
#pragma unroll
    for (int c = 0; c < 3; ++c) bufB[(kFeat + 3 + c) * kThreads + tid] = wo[c];

    float acc[3] = { 0.0f, 0.0f, 0.0f };
    for (int l = 0; l < lights.n; ++l) {
        float wiw[3], E[3], wi[3], rgb[3];
        light_sample(lights.light[l], pos.x, pos.y, pos.z, wiw, E);
        to_local(f, wiw[0], wiw[1], wiw[2], wi);
#pragma unroll
        for (int c = 0; c < 3; ++c) bufB[(kFeat + c) * kThreads + tid] = wi[c];
        mlp_b(net, lay, bufA, bufB, bufC, tid, rgb);
        const float cs = fmaxf(wi[2], 0.0f);
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[c] = fmaf(rgb[c] * E[c], cs, acc[c]);
    }
    if (live) {
        const bool bg = mat < 0;
        out[3 * p + 0] = bg ? 0.0f : acc[0];
        out[3 * p + 1] = bg ? 0.0f : acc[1];
        out[3 * p + 2] = bg ? 0.0f : acc[2];
    }
}

static size_t fp32_smem(const NetParams& net)
{
    int k = net.H;
    if (net.L + 3 > k) k = net.L + 3;
    if (kFeat + 6 > k) k = kFeat + 6;
    return (size_t)3 * k * kThreads * sizeof(float);
}

cudaError_t init_fp32()
{
    cudaError_t e = cudaFuncSetAttribute(eval_fp32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 3 * 128 * kThreads * 4);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(shade_fp32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 3 * 128 * kThreads * 4);
}

cudaError_t launch_eval_fp32(const NetParams& net, const nbsdf_query* q, const float* frames, int64_t n, float* rgb,
                             cudaStream_t s)
{
    const unsigned grid = (unsigned)((n + kThreads - 1) / kThreads);
    eval_fp32_kernel<<<grid, kThreads, fp32_smem(net), s>>>(net, q, frames, n, rgb);
    return cudaGetLastError();
}

cudaError_t launch_shade_fp32(const NetParams& net, const FrameParams& fr, const LightParams& lights, float* out,
                              cudaStream_t s)
{
    const unsigned grid = (unsigned)((fr.n_pixels + kThreads - 1) / kThreads);
    shade_fp32_kernel<<<grid, kThreads, fp32_smem(net), s>>>(net, fr, lights, out);
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
