// nbsdf_fp32.cu -- fp32 CUDA-core variant of the fused decoder (NBSDF_PREC_FP32): plain FMA, no TF32, no tensor
// cores.  A CTA owns a tile of 256 (H = 32) or 128 (H >= 64) queries; activations live in shared memory as
// [k][query] rows and every layer is a register-tiled product (4 x 8 outputs per thread at H = 64).  For H <= 64 the
// layer's transposed weights + bias sit in a shared-memory buffer (<= 16.6 KB) that is refilled layer by layer: the next
// layer's chunk is fetched into registers BEFORE the current layer's FMAs and stored after them, so the inner loop is
// LDS.128 + FMA only (round 2 read the weights with warp-uniform LDG from L1 and stalled on them: long-scoreboard 55 %
// of samples).  H = 128 keeps the L1 path (its 196 KB of activations leave no room).  Accumulation runs over k in index
// order, like the oracle's definition, in fp32.
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
template <int TQ, int TN, bool kRelu, bool kSmemW>
__device__ __forceinline__ void dense_layer(const float* __restrict__ Wt, const float* __restrict__ b, int K,
                                            const float* in, float* out)
{
    constexpr int Q = 32 * TQ, N = kWarps * TN;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int q0 = lane * TQ, n0 = warp * TN;
    float acc[TN][TQ];
#pragma unroll
    for (int j = 0; j < TN; ++j) {
        const float bj = kSmemW ? b[n0 + j] : __ldg(b + n0 + j);
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
            const float4* wp = reinterpret_cast<const float4*>(Wt + (size_t)k * N + n0 + j);
            const float4 v = kSmemW ? *wp : __ldg(wp);
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

// Per-layer weight staging (kStage): chunk l = blob[w_off[l], w_off[l+1]) = transposed weights followed by the bias, a
// multiple of 4 floats.  fetch(l) starts the global loads of chunk l into PF float4 registers per thread; commit() stores
// them into the shared buffer (the caller has synchronised: nobody still reads the previous chunk) -- the loads'
// latency passes under the FMAs of the layer in between.  Without kStage both are no-ops and W()/B() point into the blob.
template <bool kStage, int PF>
struct WStage {
    float* wbuf;
    const float* blob;
    Fp32Layout lay;
    float4 pre[PF];
    int cur;                                              // layer whose chunk is (being put) in wbuf
    static constexpr bool kStaged = kStage;

    __device__ __forceinline__ uint32_t chunk_end(int l) const { return l == 5 ? lay.total : lay.w_off[l + 1]; }
    __device__ __forceinline__ void fetch(int l)
    {
        if constexpr (kStage) {
            const float4* src = reinterpret_cast<const float4*>(blob + lay.w_off[l]);
            const int n4 = (int)((chunk_end(l) - lay.w_off[l]) >> 2);
#pragma unroll
            for (int j = 0; j < PF; ++j) {
                const int i = threadIdx.x + j * kThreads;
                if (i < n4) pre[j] = __ldg(src + i);
            }
            cur = l;
        }
    }
    __device__ __forceinline__ void commit()
    {
        if constexpr (kStage) {
            const int n4 = (int)((chunk_end(cur) - lay.w_off[cur]) >> 2);
#pragma unroll
            for (int j = 0; j < PF; ++j) {
                const int i = threadIdx.x + j * kThreads;
                if (i < n4) reinterpret_cast<float4*>(wbuf)[i] = pre[j];
            }
        }
    }
    __device__ __forceinline__ const float* W(int l) const { return kStage ? wbuf : blob + lay.w_off[l]; }
    __device__ __forceinline__ const float* B(int l) const { return kStage ? wbuf + (lay.b_off[l] - lay.w_off[l]) : blob + lay.b_off[l]; }
    // after a layer: everyone has finished reading wbuf -> store the prefetched chunk -> visible to everyone
    __device__ __forceinline__ void turn()
    {
        __syncthreads();
        if constexpr (kStage) {
            commit();
            __syncthreads();
        }
    }
};

// MLP-A: x = [z, u', v', lf] in bufA -> feat in bufB rows [0, F).  On entry wbuf holds chunk 0; on exit chunk 3.
template <int TQ, int TN, class WS>
__device__ __forceinline__ void mlp_a(const NetParams& net, WS& ws, float* bufA, float* bufB)
{
    constexpr bool S = WS::kStaged;
    ws.fetch(1);
    dense_layer<TQ, TN, true, S>(ws.W(0), ws.B(0), net.L + 3, bufA, bufB);
    ws.turn();
    ws.fetch(2);
    dense_layer<TQ, TN, true, S>(ws.W(1), ws.B(1), net.H, bufB, bufA);
    ws.turn();
    ws.fetch(3);
    dense_layer<TQ, kFeat / kWarps, false, S>(ws.W(2), ws.B(2), net.H, bufA, bufB);
    ws.turn();
}

// MLP-B: y = [feat, wi, wo] in bufB rows [0, F+6) -> rgb of query q (threads q < 32 TQ); bufB is preserved.
// On entry wbuf holds chunk 3; `again`: another MLP-B follows (next light), so chunk 3 is put back at the end -- the
// caller's __syncthreads() before that next MLP-B makes it visible.
template <int TQ, int TN, class WS>
__device__ __forceinline__ void mlp_b(const NetParams& net, WS& ws, float* bufA, float* bufB, float* bufC, float rgb[3], bool again)
{
    constexpr int Q = 32 * TQ;
    constexpr bool S = WS::kStaged;
    const float* w = net.w32;
    ws.fetch(4);
    dense_layer<TQ, TN, true, S>(ws.W(3), ws.B(3), kFeat + 6, bufB, bufA);
    ws.turn();
    if (again) ws.fetch(3);
    dense_layer<TQ, TN, true, S>(ws.W(4), ws.B(4), net.H, bufA, bufC);
    __syncthreads();
    if (again) ws.commit();
    const int qi = threadIdx.x;
    if (qi < Q) {
        const float* W6 = w + ws.lay.w_off[5];
        const float* b6 = w + ws.lay.b_off[5];
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

// largest chunk (weights + bias, floats) of layers 0..4: what the staging buffer must hold
__host__ __device__ inline uint32_t fp32_chunk_max(const Fp32Layout& lay)
{
    uint32_t m = 0;
    for (int l = 0; l < 5; ++l) m = lay.w_off[l + 1] - lay.w_off[l] > m ? lay.w_off[l + 1] - lay.w_off[l] : m;
    return m;
}

template <int TQ, int TN>
struct Fp32Cfg {
    static constexpr bool kStage = TN <= 8;                       // H <= 64
    static constexpr int kPF = TN == 8 ? 5 : 2;                   // float4 per thread of the largest chunk: H=64: 1040/256, H=32: 312/256
};

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
    WStage<Fp32Cfg<TQ, TN>::kStage, Fp32Cfg<TQ, TN>::kPF> ws;
    ws.wbuf = bufC + kmax * Q;
    ws.blob = net.w32;
    ws.lay = lay;
    ws.fetch(0);                                                  // in flight under the input assembly

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
    ws.commit();
    __syncthreads();
    mlp_a<TQ, TN>(net, ws, bufA, bufB);
    if (mine) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            bufB[(kFeat + c) * Q + tid] = wi[c];
            bufB[(kFeat + 3 + c) * Q + tid] = wo[c];
        }
    }
    __syncthreads();
    float rgb[3] = { 0.0f, 0.0f, 0.0f };
    mlp_b<TQ, TN>(net, ws, bufA, bufB, bufC, rgb, false);
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
    WStage<Fp32Cfg<TQ, TN>::kStage, Fp32Cfg<TQ, TN>::kPF> ws;
    ws.wbuf = bufC + kmax * Q;
    ws.blob = net.w32;
    ws.lay = lay;
    ws.fetch(0);

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
    ws.commit();
    __syncthreads();
    mlp_a<TQ, TN>(net, ws, bufA, bufB);      // once per pixel (the spatial feature does not depend on wi/wo)
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
        mlp_b<TQ, TN>(net, ws, bufA, bufB, bufC, rgb, l + 1 < lights.n);
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

template <int TQ, int TN>
static size_t fp32_smem(const NetParams& net)
{
    const size_t act = (size_t)3 * kmax_of(net.L, net.H) * 32 * TQ * sizeof(float);
    return act + (Fp32Cfg<TQ, TN>::kStage ? fp32_chunk_max(fp32_layout(net.L, net.H)) * sizeof(float) : 0);
}

// H = 32: 8 queries x 4 outputs per thread; H = 64: 4 x 8 (128-query tiles: 96 KB + 16.3 KB of staged weights, two CTAs
// per SM still fit: 2 x (112.3 + 1) KB <= 228 KB -- two CTAs measured 16 % faster than 8 x 8 with one CTA per SM); H = 128: 4 x 16 (a 128-query tile keeps three buffers in 196 KB)
#ifndef NBSDF_FP32_TQ64
#define NBSDF_FP32_TQ64 4
#endif
#define NBSDF_FP32_DISPATCH(CALL)                                  \
    switch (net.H) {                                               \
    case 32: { constexpr int TQ = 8, TN = 4; CALL; } break;        \
    case 64: { constexpr int TQ = NBSDF_FP32_TQ64, TN = 8; CALL; } break; \
    case 128: { constexpr int TQ = 4, TN = 16; CALL; } break;      \
    default: return cudaErrorInvalidValue;                         \
    }

cudaError_t init_fp32()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](const void* k) { if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024); };
    set((const void*)eval_fp32_kernel<8, 4>); set((const void*)eval_fp32_kernel<NBSDF_FP32_TQ64, 8>); set((const void*)eval_fp32_kernel<4, 16>);
    set((const void*)shade_fp32_kernel<8, 4>); set((const void*)shade_fp32_kernel<NBSDF_FP32_TQ64, 8>); set((const void*)shade_fp32_kernel<4, 16>);
    return e;
}

cudaError_t launch_eval_fp32(const NetParams& net, const nbsdf_query* q, const float* frames, int64_t n, float* rgb,
                             cudaStream_t s)
{
    NBSDF_FP32_DISPATCH((eval_fp32_kernel<TQ, TN><<<(unsigned)((n + 32 * TQ - 1) / (32 * TQ)), kThreads, fp32_smem<TQ, TN>(net), s>>>(
        net, q, frames, n, rgb)))
    return cudaGetLastError();
}

cudaError_t launch_shade_fp32(const NetParams& net, const FrameParams& fr, const LightParams& lights, float* out,
                              cudaStream_t s)
{
    NBSDF_FP32_DISPATCH((shade_fp32_kernel<TQ, TN><<<(unsigned)((fr.n_pixels + 32 * TQ - 1) / (32 * TQ)), kThreads,
                                                   fp32_smem<TQ, TN>(net), s>>>(net, fr, lights, out)))
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
