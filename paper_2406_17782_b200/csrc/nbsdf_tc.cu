// nbsdf_tc.cu -- the fused tensor-core decoder for sm_100a (NBSDF_PREC_BF16 / NBSDF_PREC_FP16).
//
// One persistent CTA per SM, NWG independent warpgroups per CTA.  A warpgroup owns one tile of 128 queries
// (or pixels): thread t <-> query row t <-> TMEM lane t.  All six layers of both MLPs run as
// tcgen05.mma M=128 tiles with
//   A (activations) in TENSOR MEMORY, written by the owning thread with tcgen05.st as packed 16-bit pairs,
//   B (weights)     resident in shared memory for the whole kernel as 128-byte-swizzled K-major UMMA tiles,
//   D (accumulator) fp32 in tensor memory, read back with tcgen05.ld by the owning thread,
// so the inter-layer epilogue (ReLU, 16-bit pack) is thread-local and no activation ever touches shared
// memory or HBM.  Query tiles stream in with cp.async.bulk (TMA bulk copy) one tile ahead.  Warpgroups are not
// specialised: each alternates "issue MMAs / wait / epilogue", and the NWG warpgroups of a CTA interleave so that
// the tensor pipe, the TMEM load path and the FP32 pipes overlap across tiles.
//
// TMEM columns per warpgroup (512 / NWG available):
//   [0, H)                 accumulator (N <= H fp32 columns)
//   [H, H + H/2)           AH: hidden activations as A operand (K = H 16-bit values = H/2 columns)
//   [H + H/2, +8)          constant block (c0, c1, c2, 0, ...): A operand of the bias K step of the K = H layers
//   [H + H/2 + 8, +24)     AY: layer-1 input x = [z, u', v', lf, c] (K1p/2 columns), later y = [feat, wi, wo, c] (24 columns)
// Biases ride inside the contractions (see tc_layout in nbsdf_common.cuh): the epilogue is ReLU + 16-bit pack only.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "nbsdf_common.cuh"

#ifndef NBSDF_EPI_CHUNK
#define NBSDF_EPI_CHUNK 32
#endif
#ifndef NBSDF_NWG32_EVAL
#define NBSDF_NWG32_EVAL 7
#endif
#ifndef NBSDF_NWG64_EVAL
#define NBSDF_NWG64_EVAL 4
#endif

namespace nbsdf {

// ------------------------------------------------------------------------------------------------
// PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// Waits for the phase with the given parity.  A wait that lasts ~seconds means a broken pipeline: trap instead of
// hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    if (mbar_try_wait(bar, parity)) return;
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++spins & 0x3FFu) == 0 && clock64() - t0 > 4000000000LL) __trap();
    }
}
// 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// true in exactly one lane of a fully converged warp; keeps the surrounding code warp-uniform for the compiler,
// so that MMA operands (TMEM addresses, descriptors) live in uniform registers
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.b32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
// Programmatic dependent launch: let the next kernel on the stream start its prologue while this one runs, and
// wait for the previous kernel's memory to be visible before touching anything it may have written.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_prior_grid() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish()
{
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// D[tmem] (+)= A[tmem] * B[smem]^T, M = 128, K = 16 per instruction (SASS: UTCHMMA)
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// mbarrier arrive when all previously issued MMAs of this thread have completed (implies fence::before_thread_sync)
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// TMEM <-> registers, shape 32x32b: thread i of the warp <-> lane (base + i), register j <-> column (base + j)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r)
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
        ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
          "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* r)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}

// two fp32 -> one packed 16-bit pair (lo = even k, hi = odd k), round to nearest even, optional fused ReLU
template <bool kBf16, bool kRelu>
__device__ __forceinline__ uint32_t pack2(float lo, float hi)
{
    uint32_t d;
    if (kBf16) {
        if (kRelu) asm("cvt.rn.relu.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
        else asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    } else {
        if (kRelu) asm("cvt.rn.relu.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
        else asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    }
    return d;
}

// K-major, 128-byte-swizzled shared-memory matrix descriptor: 8-row x 128-byte atoms, 1024 bytes apart
__device__ __forceinline__ uint64_t make_b_desc(uint32_t saddr)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFFu);        // start address
    d |= (uint64_t)1 << 16;                         // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024u >> 4) << 32;              // stride byte offset between 8-row groups
    d |= (uint64_t)1 << 46;                         // descriptor version (sm_100)
    d |= (uint64_t)2 << 61;                         // SWIZZLE_128B
    return d;
}

template <bool kBf16>
__host__ __device__ constexpr uint32_t make_idesc(int N)
{
    return (1u << 4)                       // D format fp32
         | ((kBf16 ? 1u : 0u) << 7)        // A format
         | ((kBf16 ? 1u : 0u) << 10)       // B format
         | ((uint32_t)(N >> 3) << 17)      // N
         | ((uint32_t)(128 >> 4) << 24);   // M = 128;  A and B K-major, no negate, dense
}

// ------------------------------------------------------------------------------------------------
template <int L, int H, bool kBf16, int NWG, bool kShade>
struct Tc {
    static constexpr bool kMerged = !kShade && tc_eval_merged(H);    // eval, H <= 64: layers 3 and 4 are one layer
    static constexpr TcLayout kLay = tc_layout(L, H, kMerged);
    static constexpr int K1p = kLay.K1p;
    static constexpr int K4p = kLay.K4p;
    static constexpr int kThreads = NWG * 128;
    // TMEM columns of one warpgroup.  eval: x, the hidden activations and y share ONE A-operand region (each is dead
    // before the next is written); shade: y = [feat, wi, wo] must survive the light loop, so it gets its own region.
    // Merged eval adds an 8-column tail block [wi, wo, c0, c1, c2, 0...]: the last K step of the merged layer.
    static constexpr int kAw = kShade ? H / 2 : (H / 2 > 24 ? H / 2 : 24);
    static constexpr int kAccCol = 0;
    static constexpr int kAhCol = H;
    static constexpr int kAyCol = kShade ? H + H / 2 : H;
    static constexpr int kTailCol = H + kAw;
    static constexpr int kColsPerWg = kShade ? H + H / 2 + 24 : H + kAw + (kMerged ? 8 : 0);
    static constexpr int kOneCol = 504;              // CTA-wide constant block (c0, c1, c2, 0...): bias K step of the K = H layers
    static_assert(NWG * kColsPerWg <= kOneCol, "TMEM budget");
    static_assert(L % 8 == 0 && H % 32 == 0, "dims");
    static_assert(K1p <= 48 && K4p == 48, "x / y hold at most 24 columns");

    static constexpr uint32_t kLatBytes = 64 * 32 * 2;            // packed latent table, max M x max L
    static constexpr uint32_t kStageBytes = 128 * sizeof(nbsdf_query);

    __host__ __device__ static constexpr uint32_t wimg_bytes() { return kLay.total; }
    __host__ __device__ static constexpr uint32_t smem_bytes()
    {
        return 1024u + ((wimg_bytes() + 127u) & ~127u) + kLatBytes + NWG * kStageBytes + 256u;
    }
};

// Issues the MMAs of one layer for this warpgroup's tile and commits them to the warpgroup's mbarrier.
// Called by ONE thread.  K/16 steps in total; the first KA/16 read the A operand at a_tmem, the remaining ones
// (the bias step of the K = H layers) read the constant block at one_tmem.  d_tmem/a_tmem/one_tmem are lane-0
// TMEM addresses; w_saddr is the layer's weight tiles in shared memory.
template <bool kBf16, int K, int N, int KA>
__device__ __forceinline__ void issue_layer(uint32_t d_tmem, uint32_t a_tmem, uint32_t one_tmem, uint32_t w_saddr, uint32_t bar)
{
    constexpr uint32_t idesc = make_idesc<kBf16>(N);
    tc_fence_after();
#pragma unroll
    for (int s = 0; s < K / 16; ++s) {
        const uint32_t b = w_saddr + (uint32_t)(s >> 2) * (uint32_t)N * 128u + (uint32_t)(s & 3) * 32u;
        const uint32_t a = s < KA / 16 ? a_tmem + (uint32_t)s * 8u : one_tmem + (uint32_t)(s - KA / 16) * 8u;
        umma_ts(d_tmem, a, make_b_desc(b), idesc, s > 0 ? 1u : 0u);
    }
    umma_commit(bar);
}

// Epilogue of a hidden layer: acc (N fp32 columns, bias already inside) -> (ReLU) -> packed 16-bit pairs -> A columns.
// 64 columns are fetched per wait so that two tcgen05.ld are in flight.
template <int N, bool kRelu, bool kBf16>
__device__ __forceinline__ void epilogue_to_a(uint32_t acc_taddr, uint32_t a_taddr)
{
#if NBSDF_EPI_CHUNK == 16
#pragma unroll
    for (int c = 0; c < N; c += 16) {
        uint32_t v[16];
        tmem_ld16(acc_taddr + c, v);
        tmem_wait_ld();
        uint32_t p[8];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            p[j] = pack2<kBf16, kRelu>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
        tmem_st8(a_taddr + c / 2, p);
    }
#else
#pragma unroll
    for (int c = 0; c < N; c += 32) {
        uint32_t v[32];
        tmem_ld32(acc_taddr + c, v);
        tmem_wait_ld();
        uint32_t p[16];
#pragma unroll
        for (int j = 0; j < 16; ++j)
            p[j] = pack2<kBf16, kRelu>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
        tmem_st16(a_taddr + c / 2, p);
    }
#endif
}

// Per-thread record after input assembly (stages A1-A4)
struct Assembled {
    float up, vp, lf;
    float wi[3], wo[3];
    int material;
};

template <int L, int H, bool kBf16, int NWG, bool kShade>
__global__ void __launch_bounds__(NWG * 128, 1)
tc_kernel(NetParams net, const nbsdf_query* __restrict__ q, const float* __restrict__ frames, int64_t n,
          FrameParams fr, LightParams lights, float* __restrict__ out)
{
    using T = Tc<L, H, kBf16, NWG, kShade>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - smem_u32(smem_raw));
    constexpr uint32_t kWimgPad = (T::wimg_bytes() + 127u) & ~127u;
    const uint32_t s_wimg = base;
    const uint32_t s_lat = s_wimg + kWimgPad;
    const uint32_t s_stage = s_lat + T::kLatBytes;
    const uint32_t s_bars = s_stage + NWG * T::kStageBytes;
    const uint32_t s_tmem = s_bars + NWG * 16u;
    uint8_t* g_wimg = gbase;
    uint8_t* g_lat = g_wimg + kWimgPad;
    uint8_t* g_stage = g_lat + T::kLatBytes;
    uint32_t* g_tmem = reinterpret_cast<uint32_t*>(g_stage + NWG * T::kStageBytes + NWG * 16u);

    const int tid = threadIdx.x;
    const int t = tid & 127;               // row within the tile == TMEM lane
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);     // warp-uniform for the compiler
    const int wg = warp >> 2;
    const bool issuer = (warp & 3) == 0;   // warp 0 of each warpgroup issues its MMAs and bulk copies (one elected lane)
    constexpr TcLayout lay = T::kLay;

    // ---- prologue: weights image + packed latents -> shared memory, barriers, TMEM ----
    // The weight image is immutable after nbsdf_create, so it is fetched before the grid-dependency wait and overlaps
    // the tail of the previous kernel on the stream; everything a previous kernel or copy may write comes after it.
    pdl_launch_dependents();
    const uint32_t mma_bar = s_bars + (uint32_t)wg * 16u;
    const uint32_t q_bar = mma_bar + 8u;
    const uint32_t w_bar = s_tmem + 8u;
    if (warp == 0 && elect_one()) {
        mbar_init(w_bar, 1);
        fence_mbar_init();
        // one elected lane streams the whole image in with bulk copies; only the MMA issuers ever wait for it
        mbar_expect_tx(w_bar, T::wimg_bytes());
        constexpr uint32_t kChunk = 32768u;
        for (uint32_t off = 0; off < T::wimg_bytes(); off += kChunk) {
            const uint32_t bytes = T::wimg_bytes() - off < kChunk ? T::wimg_bytes() - off : kChunk;
            bulk_g2s(s_wimg + off, (kShade ? net.wimg_shade : net.wimg_eval) + off, bytes, w_bar);
        }
    }
    __syncwarp();
    if (issuer && elect_one()) {
        mbar_init(mma_bar, 1);
        mbar_init(q_bar, 1);
        fence_mbar_init();
    }
    __syncwarp();
    if (warp == 0) {
        tmem_alloc(s_tmem, 512);
        tmem_relinquish();
    }
    pdl_wait_prior_grid();
    {
        uint16_t* lat = reinterpret_cast<uint16_t*>(g_lat);
        for (int i = tid; i < net.M * L; i += T::kThreads) {
            const float z = __ldg(net.latents + i);
            lat[i] = kBf16 ? __bfloat16_as_ushort(__float2bfloat16_rn(z)) : __half_as_ushort(__float2half_rn(z));
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *g_tmem, 0);
    const uint32_t col0 = tmem_base + (uint32_t)(wg * T::kColsPerWg);                 // lane 0: for MMA operands
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;                      // this warp's lane quarter
    const uint32_t lane_taddr = col0 + lane_off;
    const uint32_t acc_t = lane_taddr + T::kAccCol, ah_t = lane_taddr + T::kAhCol, ay_t = lane_taddr + T::kAyCol;
    const uint32_t acc_d = col0 + T::kAccCol, ah_d = col0 + T::kAhCol, ay_d = col0 + T::kAyCol, one_d = tmem_base + T::kOneCol;

    // bias constants (c0, c1, c2) as packed pairs; the CTA-wide constant block is written once per kernel by warpgroup 0
    const uint32_t c01 = pack2<kBf16, false>(tc_bias_const(kBf16, 0), tc_bias_const(kBf16, 1));
    const uint32_t c2z = pack2<kBf16, false>(tc_bias_const(kBf16, 2), 0.0f);
    if (wg == 0) {
        uint32_t ones[8] = { c01, c2z, 0u, 0u, 0u, 0u, 0u, 0u };
        tmem_st8(tmem_base + lane_off + T::kOneCol, ones);
        tmem_wait_st();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    uint32_t w_s[6];
#pragma unroll
    for (int l = 0; l < 6; ++l) w_s[l] = s_wimg + (l < lay.n_layers ? lay.w_off[l] : 0u);

    const int64_t n_items = kShade ? fr.n_pixels : n;
    const int64_t n_tiles = (n_items + 127) / 128;
    const int64_t stride = (int64_t)gridDim.x * NWG;
    const int64_t first = (int64_t)blockIdx.x * NWG + wg;
    uint32_t mma_phase = 0, q_phase = 0;
    bool weights_ready = false;
    const uint32_t my_stage = s_stage + (uint32_t)wg * T::kStageBytes;
    const uint8_t* my_stage_g = g_stage + (size_t)wg * T::kStageBytes;

    auto tile_is_bulk = [&](int64_t tile) { return !kShade && tile < n_tiles && (tile + 1) * 128 <= n_items; };
    if (issuer && tile_is_bulk(first) && elect_one()) {
        mbar_expect_tx(q_bar, T::kStageBytes);
        bulk_g2s(my_stage, q + first * 128, T::kStageBytes, q_bar);
    }
    __syncwarp();

    // One MMA round: publish the A operand this thread just wrote, let the issuer lane issue, wait for completion.
    auto publish = [&]() {
        tmem_wait_st();
        tc_fence_before();
        named_bar_sync(1 + wg, 128);
    };
    auto await_mma = [&]() {
        mbar_wait(mma_bar, mma_phase);
        mma_phase ^= 1u;
        tc_fence_after();
    };

    // shade: this thread's G-buffer texel of the NEXT tile is requested one tile ahead and lands in registers while the
    // current tile computes (52 B/pixel, perfectly coalesced float4 planes)
    float4 pf_pos = make_float4(0.f, 0.f, 0.f, 1.f), pf_nu = make_float4(0.f, 0.f, 1.f, 0.f), pf_tv = make_float4(1.f, 0.f, 0.f, 0.f);
    int pf_mat = -1;
    auto gbuf_request = [&](int64_t tile) {
        const int64_t it = tile * 128 + t;
        pf_pos = make_float4(0.f, 0.f, 0.f, 1.f); pf_nu = make_float4(0.f, 0.f, 1.f, 0.f); pf_tv = make_float4(1.f, 0.f, 0.f, 0.f);
        pf_mat = -1;
        if (tile < n_tiles && it < n_items) {
            pf_pos = __ldg(fr.pos_fp + it); pf_nu = __ldg(fr.nrm_u + it); pf_tv = __ldg(fr.tan_v + it);
            pf_mat = __ldg(fr.material + it);
        }
    };
    if (kShade) gbuf_request(first);

    for (int64_t tile = first; tile < n_tiles; tile += stride) {
        const int64_t item = tile * 128 + t;
        const bool live = item < n_items;

        // ---- stages A1-A4: fetch + assemble ----
        Assembled a;
        a.up = a.vp = 0.0f; a.lf = 0.0f; a.material = -1;
        a.wi[0] = a.wi[1] = 0.0f; a.wi[2] = 1.0f; a.wo[0] = a.wo[1] = 0.0f; a.wo[2] = 1.0f;
        float px = 0.0f, py = 0.0f, pz = 0.0f;
        Frame f;
        if (!kShade) {
            nbsdf_query rec;
            rec.u = rec.v = 0.0f; rec.footprint = 1.0f; rec.material = -1;
            rec.wi[0] = rec.wi[1] = 0.0f; rec.wi[2] = 1.0f; rec.wo[0] = rec.wo[1] = 0.0f; rec.wo[2] = 1.0f;
            if (tile_is_bulk(tile)) {
                mbar_wait(q_bar, q_phase);
                q_phase ^= 1u;
                const uint2* r2 = reinterpret_cast<const uint2*>(my_stage_g + t * sizeof(nbsdf_query));
                uint2 w0 = r2[0], w1 = r2[1], w2 = r2[2], w3 = r2[3], w4 = r2[4];
                rec.u = __uint_as_float(w0.x); rec.v = __uint_as_float(w0.y);
                rec.footprint = __uint_as_float(w1.x); rec.material = (int)w1.y;
                rec.wi[0] = __uint_as_float(w2.x); rec.wi[1] = __uint_as_float(w2.y); rec.wi[2] = __uint_as_float(w3.x);
                rec.wo[0] = __uint_as_float(w3.y); rec.wo[1] = __uint_as_float(w4.x); rec.wo[2] = __uint_as_float(w4.y);
            } else if (live) {
                const uint2* r2 = reinterpret_cast<const uint2*>(q + item);
                uint2 w0 = __ldg(r2), w1 = __ldg(r2 + 1), w2 = __ldg(r2 + 2), w3 = __ldg(r2 + 3), w4 = __ldg(r2 + 4);
                rec.u = __uint_as_float(w0.x); rec.v = __uint_as_float(w0.y);
                rec.footprint = __uint_as_float(w1.x); rec.material = (int)w1.y;
                rec.wi[0] = __uint_as_float(w2.x); rec.wi[1] = __uint_as_float(w2.y); rec.wi[2] = __uint_as_float(w3.x);
                rec.wo[0] = __uint_as_float(w3.y); rec.wo[1] = __uint_as_float(w4.x); rec.wo[2] = __uint_as_float(w4.y);
            }
            a.up = wrap01(rec.u); a.vp = wrap01(rec.v); a.lf = log_footprint<true>(rec.footprint);
            a.material = rec.material;
#pragma unroll
            for (int c = 0; c < 3; ++c) { a.wi[c] = rec.wi[c]; a.wo[c] = rec.wo[c]; }
            if (frames != nullptr && live) {
                const float2* fp2 = reinterpret_cast<const float2*>(frames + 6 * item);
                const float2 f0 = __ldg(fp2), f1 = __ldg(fp2 + 1), f2 = __ldg(fp2 + 2);
                f = make_frame(f0.x, f0.y, f1.x, f1.y, f2.x, f2.y);
                to_local(f, rec.wi[0], rec.wi[1], rec.wi[2], a.wi);
                to_local(f, rec.wo[0], rec.wo[1], rec.wo[2], a.wo);
            }
        } else {
            const float4 pos = pf_pos, nu = pf_nu, tv = pf_tv;
            a.material = pf_mat;
            gbuf_request(tile + stride);
            px = pos.x; py = pos.y; pz = pos.z;
            f = make_frame(nu.x, nu.y, nu.z, tv.x, tv.y, tv.z);
            float vx = fr.cam[0] - px, vy = fr.cam[1] - py, vz = fr.cam[2] - pz;
            const float inv = rsqrtf(vx * vx + vy * vy + vz * vz);
            to_local(f, vx * inv, vy * inv, vz * inv, a.wo);
            a.up = wrap01(nu.w); a.vp = wrap01(tv.w); a.lf = log_footprint<true>(pos.w);
        }

        // ---- layer-1 operand x = [z, u', v', lf, 0...] -> AY ----
        {
            const int m = a.material < 0 ? 0 : a.material;
            uint32_t x[T::K1p / 2];
            const uint4* zrow = reinterpret_cast<const uint4*>(g_lat + (size_t)m * L * 2);
#pragma unroll
            for (int i = 0; i < L / 8; ++i) {
                const uint4 z4 = zrow[i];
                x[4 * i] = z4.x; x[4 * i + 1] = z4.y; x[4 * i + 2] = z4.z; x[4 * i + 3] = z4.w;
            }
            x[L / 2] = pack2<kBf16, false>(a.up, a.vp);
            x[L / 2 + 1] = pack2<kBf16, false>(a.lf, tc_bias_const(kBf16, 0));
            x[L / 2 + 2] = pack2<kBf16, false>(tc_bias_const(kBf16, 1), tc_bias_const(kBf16, 2));
#pragma unroll
            for (int i = L / 2 + 3; i < T::K1p / 2; ++i) x[i] = 0u;
#pragma unroll
            for (int i = 0; i < T::K1p / 2; i += 8) tmem_st8(ay_t + i, x + i);
            if constexpr (T::kMerged) {   // tail block of the merged layer: [wi, wo, c0, c1, c2, 0...]
                uint32_t y[8];
                y[0] = pack2<kBf16, false>(a.wi[0], a.wi[1]);
                y[1] = pack2<kBf16, false>(a.wi[2], a.wo[0]);
                y[2] = pack2<kBf16, false>(a.wo[1], a.wo[2]);
                y[3] = c01;
                y[4] = c2z;
#pragma unroll
                for (int i = 5; i < 8; ++i) y[i] = 0u;
                tmem_st8(lane_taddr + T::kTailCol, y);
            }
        }

        // ---- MLP-A (B1-B3) ----
        publish();                            // every thread has consumed its staged record and stored x
        if (issuer) {
            if (elect_one()) {
                const int64_t next = tile + stride;
                if (tile_is_bulk(next)) {          // stream the next tile's records in while this one computes
                    mbar_expect_tx(q_bar, T::kStageBytes);
                    bulk_g2s(my_stage, q + next * 128, T::kStageBytes, q_bar);
                }
                if (!weights_ready) mbar_wait(w_bar, 0);
                issue_layer<kBf16, T::K1p, H, T::K1p>(acc_d, ay_d, one_d, w_s[0], mma_bar);
            }
            weights_ready = true;
            __syncwarp();
        }
        await_mma();

        epilogue_to_a<H, true, kBf16>(acc_t, ah_t);
        publish();
        if (issuer) {
            if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[1], mma_bar);
            __syncwarp();
        }
        await_mma();
        epilogue_to_a<H, true, kBf16>(acc_t, ah_t);
        float rad[3] = { 0.0f, 0.0f, 0.0f };
        // last two layers of MLP-B + softplus (B5-B7); g1 has just been published as the A operand
        auto finish_mlp_b = [&](uint32_t w5, uint32_t w6, const float E[3], float cs) {
            if (issuer) {
                if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w5, mma_bar);
                __syncwarp();
            }
            await_mma();
            epilogue_to_a<H, true, kBf16>(acc_t, ah_t);
            publish();
            if (issuer) {
                if (elect_one()) issue_layer<kBf16, H + 16, 16, H>(acc_d, ah_d, one_d, w6, mma_bar);
                __syncwarp();
            }
            await_mma();
            uint32_t o[4];
            tmem_ld4(acc_t, o);
            tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float v = softplus<true>(__uint_as_float(o[c]));
                rad[c] = kShade ? fmaf(v * E[c], cs, rad[c]) : v;
            }
        };
        if constexpr (T::kMerged) {
            // ---- merged layers 3+4 (B3-B4): (W4f W3) h2 + W4a [wi, wo] + (W4f b3 + b4); K = H from AH + tail block ----
            publish();
            if (issuer) {
                if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, col0 + T::kTailCol, w_s[2], mma_bar);
                __syncwarp();
            }
            await_mma();
            epilogue_to_a<H, true, kBf16>(acc_t, ah_t);
            publish();
            const float E1[3] = { 1.0f, 1.0f, 1.0f };
            finish_mlp_b(w_s[3], w_s[4], E1, 1.0f);
        } else {
            publish();
            if (issuer) {
                if (elect_one()) issue_layer<kBf16, H + 16, kFeat, H>(acc_d, ah_d, one_d, w_s[2], mma_bar);
                __syncwarp();
            }
            await_mma();
            epilogue_to_a<kFeat, false, kBf16>(acc_t, ay_t);      // feat (linear) -> AY columns [0, 16)

            // ---- MLP-B (B4-B7), once per query / once per light (C1-C3) ----
            const int n_rounds = kShade ? lights.n : 1;
            for (int l = 0; l < n_rounds; ++l) {
                float E[3] = { 1.0f, 1.0f, 1.0f };
                float cs = 1.0f;
                if (kShade) {
                    float wiw[3];
                    light_sample(lights.light[l], px, py, pz, wiw, E);
                    to_local(f, wiw[0], wiw[1], wiw[2], a.wi);
                    cs = fmaxf(a.wi[2], 0.0f);
                }
                uint32_t y[8];
                y[0] = pack2<kBf16, false>(a.wi[0], a.wi[1]);
                y[1] = pack2<kBf16, false>(a.wi[2], a.wo[0]);
                y[2] = pack2<kBf16, false>(a.wo[1], a.wo[2]);
                y[3] = c01;
                y[4] = c2z;
#pragma unroll
                for (int i = 5; i < 8; ++i) y[i] = 0u;
                tmem_st8(ay_t + 16, y);
                publish();
                if (issuer) {
                    if (elect_one()) issue_layer<kBf16, T::K4p, H, T::K4p>(acc_d, ay_d, one_d, w_s[3], mma_bar);
                    __syncwarp();
                }
                await_mma();
                epilogue_to_a<H, true, kBf16>(acc_t, ah_t);
                publish();
                finish_mlp_b(w_s[4], w_s[5], E, cs);
            }
        }
        if (live) {
            const bool bg = a.material < 0;
            out[3 * item + 0] = bg ? 0.0f : rad[0];
            out[3 * item + 1] = bg ? 0.0f : rad[1];
            out[3 * item + 2] = bg ? 0.0f : rad[2];
        }
    }

    // ---- teardown ----
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, 512);
}

// ------------------------------------------------------------------------------------------------
template <int L, int H, bool kBf16, bool kShade>
static cudaError_t launch_one(const NetParams& net, int num_sms, const nbsdf_query* q, const float* frames, int64_t n,
                              const FrameParams& fr, const LightParams& lights, float* out, cudaStream_t s, bool init_only)
{
    constexpr int NWG = H == 128 ? 2 : (H == 32 ? (kShade ? 6 : NBSDF_NWG32_EVAL) : (kShade ? 4 : NBSDF_NWG64_EVAL));
    using T = Tc<L, H, kBf16, NWG, kShade>;
    auto kern = tc_kernel<L, H, kBf16, NWG, kShade>;
    if (init_only) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::smem_bytes());
    const int64_t n_items = kShade ? fr.n_pixels : n;
    const int64_t tiles = (n_items + 127) / 128;
    int64_t grid = (tiles + NWG - 1) / NWG;
    if (grid > num_sms) grid = num_sms;
    if (grid < 1) grid = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(NWG * 128);
    cfg.dynamicSmemBytes = T::smem_bytes();
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // overlap our prologue with the previous kernel's tail
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, net, q, frames, n, fr, lights, out);
}

template <bool kShade>
static cudaError_t dispatch(const NetParams& net, int precision, int num_sms, const nbsdf_query* q, const float* frames,
                            int64_t n, const FrameParams& fr, const LightParams& lights, float* out, cudaStream_t s,
                            bool init_only)
{
    const bool bf = precision == NBSDF_PREC_BF16;
#define NBSDF_CASE(LL, HH)                                                                                             \
    if (net.L == LL && net.H == HH)                                                                                    \
        return bf ? launch_one<LL, HH, true, kShade>(net, num_sms, q, frames, n, fr, lights, out, s, init_only)       \
                  : launch_one<LL, HH, false, kShade>(net, num_sms, q, frames, n, fr, lights, out, s, init_only);
    NBSDF_CASE(8, 32) NBSDF_CASE(16, 32) NBSDF_CASE(32, 32)
    NBSDF_CASE(8, 64) NBSDF_CASE(16, 64) NBSDF_CASE(32, 64)
    NBSDF_CASE(8, 128) NBSDF_CASE(16, 128) NBSDF_CASE(32, 128)
#undef NBSDF_CASE
    return cudaErrorInvalidValue;
}

cudaError_t init_tc(int L, int H)
{
    NetParams net{};
    net.L = L; net.H = H;
    FrameParams fr{};
    LightParams lt{};
    for (int prec = NBSDF_PREC_BF16; prec <= NBSDF_PREC_FP16; ++prec) {
        cudaError_t e = dispatch<false>(net, prec, 1, nullptr, nullptr, 0, fr, lt, nullptr, 0, true);
        if (e != cudaSuccess) return e;
        e = dispatch<true>(net, prec, 1, nullptr, nullptr, 0, fr, lt, nullptr, 0, true);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_eval_tc(const NetParams& net, int precision, int num_sms, const nbsdf_query* q, const float* frames,
                           int64_t n, float* rgb, cudaStream_t s)
{
    FrameParams fr{};
    LightParams lt{};
    return dispatch<false>(net, precision, num_sms, q, frames, n, fr, lt, rgb, s, false);
}

cudaError_t launch_shade_tc(const NetParams& net, int precision, int num_sms, const FrameParams& fr,
                            const LightParams& lights, float* out, cudaStream_t s)
{
    return dispatch<true>(net, precision, num_sms, nullptr, nullptr, 0, fr, lights, out, s, false);
}

}  // namespace nbsdf
