// nbsdf_tc.cu -- the fused tensor-core decoder for sm_100a (NBSDF_PREC_BF16 / NBSDF_PREC_FP16).
//
// One persistent CTA per SM, NWG independent warpgroups per CTA.  A warpgroup owns one tile of 128 queries
// (or pixels): thread t <-> query row t <-> TMEM lane t.  All six layers of both MLPs run as
// tcgen05.mma M=128 tiles with
//   A (activations) in TENSOR MEMORY, written by the owning thread with tcgen05.st as packed 16-bit pairs,
//   B (weights)     resident in shared memory for the whole kernel as 128-byte-swizzled K-major UMMA tiles,
//   D (accumulator) fp32 in tensor memory, read back with tcgen05.ld by the owning thread,
// so the inter-layer epilogue (ReLU, 16-bit pack) is thread-local and no activation ever touches shared
// memory or HBM.  Query tiles stream in with cp.async.bulk (TMA bulk copy) three tiles ahead.  The CTA is warp-
// specialised: warps [0, 4 NWG) are the row owners (input assembly, epilogues, output), and one extra MMA-issuer warp
// per warpgroup issues that warpgroup's tcgen05.mma chains and its bulk copies; the NWG tiles in flight interleave so
// that the tensor pipe, the TMEM load path and the ALU pipes overlap across tiles.
//
// TMEM columns per warpgroup (504 / NWG available; the last 8 hold the CTA-wide bias-constant block), see struct Tc:
//   [0, H)                 accumulator (N <= H fp32 columns)
//   [H, H + kAw)           AH: hidden activations as A operand (K = H 16-bit values = H/2 columns); eval: also x / y
//   shade:  [H + H/2, +24) AY: x = [z, u', v', lf, c] (K1p/2 columns), later y = [feat, wi, wo, c] (24 columns)
//   merged eval: +8        tail block [wi, wo, c0, c1, c2, 0...]: last K step of the merged layer;  +K1p/2: x (kXDirect)
// Biases ride inside the contractions (see tc_layout in nbsdf_common.cuh): the epilogue is ReLU + 16-bit pack only.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "nbsdf_common.cuh"
#include "nbsdf_probe.cuh"
#include "nbsdf_tc_ptx.cuh"

#ifndef NBSDF_NWG32_EVAL
#define NBSDF_NWG32_EVAL 6
#endif
#ifndef NBSDF_NWG64_EVAL
#define NBSDF_NWG64_EVAL 4
#endif
#ifndef NBSDF_NWG64_SHADE
#define NBSDF_NWG64_SHADE 4
#endif

namespace nbsdf {

// ------------------------------------------------------------------------------------------------
template <int L, int H, bool kBf16, int NWG, bool kShade>
struct Tc {
    static constexpr bool kMerged = !kShade && tc_eval_merged(H);    // eval, H <= 64: layers 3 and 4 are one layer
    static constexpr TcLayout kLay = tc_layout(L, H, kMerged);
    static constexpr int K1p = kLay.K1p;
    static constexpr int K4p = kLay.K4p;
    // Warps [0, 4 NWG) are the warpgroups that own tile rows; then one MMA-issuer warp per warpgroup, padded to whole
    // warpgroups so that setmaxnreg can move the issuers' registers to the row owners.
    static constexpr int kIssuerWarps = (NWG + 3) / 4 * 4;
    static constexpr int kThreads = NWG * 128 + kIssuerWarps * 32;
    static constexpr int kIssuerRegs = 56;
    static constexpr int kBaseRegs = 65536 / kThreads / 8 * 8 > 248 ? 248 : 65536 / kThreads / 8 * 8;      // what ptxas is told
    // only what the issuer warps give back is available to setmaxnreg.inc (not the register file's unallocated rest)
    static constexpr int kOwnerRegsRaw = kBaseRegs + kIssuerWarps * 32 * (kBaseRegs - kIssuerRegs) / (NWG * 128) / 8 * 8;
    static constexpr int kOwnerRegs = kOwnerRegsRaw > 248 ? 248 : kOwnerRegsRaw;
    static_assert(kThreads <= 1024, "CTA size");
    static constexpr bool kTwoLoads = kOwnerRegs >= (kShade ? 150 : 100);         // epilogue register budget (see epilogue_to_a)
    // TMEM columns of one warpgroup.  eval: x, the hidden activations and y share ONE A-operand region (each is dead
    // before the next is written); shade: y = [feat, wi, wo] must survive the light loop, so it gets its own region.
    // Merged eval adds an 8-column tail block [wi, wo, c0, c1, c2, 0...]: the last K step of the merged layer.
    static constexpr int kAw = kShade ? H / 2 : (H / 2 > 24 ? H / 2 : 24);
    static constexpr int kAccCol = 0;
    static constexpr int kAhCol = H;
    static constexpr int kAyCol = kShade ? H + H / 2 : H;
    static constexpr int kTailCol = H + kAw;
    // merged eval, when the columns are there: x gets a region of its own (read by layer 1 only), so that the input
    // assembly of the next tile stores x and the tail block straight to TMEM and a tile starts without any store
    static constexpr bool kXDirect = kMerged && NWG * (H + kAw + 8 + K1p / 2) <= 504;
    static constexpr int kXCol = H + kAw + 8;
    static constexpr int kColsPerWg = kShade ? H + H / 2 + 24 : H + kAw + (kMerged ? 8 : 0) + (kXDirect ? K1p / 2 : 0);
    static constexpr int kOneCol = 504;              // CTA-wide constant block (c0, c1, c2, 0...): bias K step of the K = H layers
    static_assert(NWG * kColsPerWg <= kOneCol, "TMEM budget");
    static_assert(L % 8 == 0 && H % 32 == 0, "dims");
    static_assert(K1p <= 48 && K4p == 48, "x / y hold at most 24 columns");

    static constexpr uint32_t kLatBytes = 64 * 32 * 2;            // packed latent table, max M x max L
    static constexpr uint32_t kStageBytes = 128 * sizeof(nbsdf_query);      // one tile of query records ...
    static constexpr uint32_t kFrameBytes = 128 * 6 * sizeof(float);         // ... and of per-query frames behind it
    static constexpr uint32_t kStageStride = kStageBytes + kFrameBytes;      // 8192
    static constexpr uint32_t kStages = 2;                        // staging buffers per warpgroup

    __host__ __device__ static constexpr uint32_t wimg_bytes() { return kLay.total; }
    __host__ __device__ static constexpr uint32_t smem_bytes()
    {
        return 1024u + ((wimg_bytes() + 127u) & ~127u) + kLatBytes + NWG * kStages * kStageStride + NWG * 32u + 64u;
    }
};

// Epilogue of a hidden layer: acc (N fp32 columns, bias already inside) -> (ReLU) -> packed 16-bit pairs -> A columns.
// kTwoLoads: 64 columns (two tcgen05.ld) are requested per wait, so the second load's latency hides behind the
// first's; costs 32 more live registers.
template <int N, bool kRelu, bool kBf16, bool kTwoLoads = true>
__device__ __forceinline__ void epilogue_to_a(uint32_t acc_taddr, uint32_t a_taddr)
{
    if constexpr (kTwoLoads && N % 64 == 0) {
#pragma unroll
        for (int c = 0; c < N; c += 64) {
            uint32_t v[32], w[32];
            tmem_ld32(acc_taddr + c, v);
            tmem_ld32(acc_taddr + c + 32, w);
            tmem_wait_ld();
            uint32_t p[16];
#pragma unroll
            for (int j = 0; j < 16; ++j)
                p[j] = pack2<kBf16, kRelu>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
            tmem_st16(a_taddr + c / 2, p);
#pragma unroll
            for (int j = 0; j < 16; ++j)
                p[j] = pack2<kBf16, kRelu>(__uint_as_float(w[2 * j]), __uint_as_float(w[2 * j + 1]));
            tmem_st16(a_taddr + c / 2 + 16, p);
        }
    } else {
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
    }
}

// The kernel.  Per warpgroup and 128-row tile the layer chain is strictly sequential
//   [operand in TMEM] -> warpgroup barrier -> one lane issues the layer's MMAs + commit -> all wait -> epilogue -> ...
// and a round trip (barrier, issue, commit, wake-up, tcgen05.ld, convert, tcgen05.st) costs about as much as the MMAs
// themselves, so the tensor pipe only stays busy if nothing else sits in that chain.  Everything that is not a layer
// therefore runs in the SHADOW of an MMA wait, one tile ahead or behind:
//   * the input assembly of the NEXT tile (stages A1-A4: staged record / G-buffer texel -> x, local wi/wo) runs
//     after one of this tile's layers has been issued and leaves its result in registers;
//   * the output of the PREVIOUS tile (stage B7 softplus, C2 accumulate, C3 store) runs after this tile's layer 1
//     has been issued; in the light loop the accumulate of light l runs after layer 4 of light l+1 has been issued
//     and the geometry of light l+1 (stage C1) after layer 5 of light l.
template <int L, int H, bool kBf16, int NWG, bool kShade>
__global__ void __launch_bounds__(Tc<L, H, kBf16, NWG, kShade>::kThreads, 1)
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
    const uint32_t s_bars = s_stage + NWG * T::kStages * T::kStageStride;
    const uint32_t s_tmem = s_bars + NWG * 32u;
    uint8_t* g_wimg = gbase;
    uint8_t* g_lat = g_wimg + kWimgPad;
    uint8_t* g_stage = g_lat + T::kLatBytes;
    uint32_t* g_tmem = reinterpret_cast<uint32_t*>(g_stage + NWG * T::kStages * T::kStageStride + NWG * 32u);

    const int tid = threadIdx.x;
    NBSDF_STAMP(tid == 0, net, 0);
    const int t = tid & 127;               // row within the tile == TMEM lane
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);     // warp-uniform for the compiler
    // warps [0, 4 NWG): the warpgroups that own tile rows; warp 4 NWG + i: the MMA / bulk-copy issuer of warpgroup i
    const bool issuer = warp >= NWG * 4;
    const int wg = issuer ? warp - NWG * 4 : warp >> 2;          // >= NWG: padding warp, idle
    constexpr TcLayout lay = T::kLay;

    // ---- prologue: weights image + packed latents -> shared memory, barriers, TMEM ----
    // The weight image is immutable after nbsdf_create, so it is fetched before the grid-dependency wait and overlaps
    // the tail of the previous kernel on the stream; everything a previous kernel or copy may write comes after it.
    pdl_launch_dependents();
    const uint32_t mma_bar = s_bars + (uint32_t)wg * 32u;
    const uint32_t q_bar = mma_bar + 8u;            // two of them: one per staging buffer
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
    if (issuer && wg < NWG && elect_one()) {
        mbar_init(mma_bar, 1);
        mbar_init(q_bar, 1);
        mbar_init(q_bar + 8u, 1);
        fence_mbar_init();
    }
    __syncwarp();
    if (warp == 0) {
        tmem_alloc(s_tmem, 512);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    NBSDF_STAMP(tid == 0, net, 1);
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *g_tmem, 0);
    const uint32_t col0 = tmem_base + (uint32_t)(wg * T::kColsPerWg);                 // lane 0: for MMA operands
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;                      // this warp's lane quarter
    const uint32_t lane_taddr = col0 + lane_off;
    const uint32_t acc_t = lane_taddr + T::kAccCol, ah_t = lane_taddr + T::kAhCol, ay_t = lane_taddr + T::kAyCol;
    const uint32_t acc_d = col0 + T::kAccCol, ah_d = col0 + T::kAhCol, ay_d = col0 + T::kAyCol, one_d = tmem_base + T::kOneCol;

    // bias constants (c0, c1, c2) as packed pairs; the CTA-wide constant block is written once per kernel by warpgroup 0
    const uint32_t c01 = pack2<kBf16, false>(tc_bias_const(kBf16, 0), tc_bias_const(kBf16, 1));
    const uint32_t c2z = pack2<kBf16, false>(tc_bias_const(kBf16, 2), 0.0f);
    if (!issuer && wg == 0) {
        uint32_t ones[8] = { c01, c2z, 0u, 0u, 0u, 0u, 0u, 0u };
        tmem_st8(tmem_base + lane_off + T::kOneCol, ones);
        tmem_wait_st();
    }
    uint32_t w_s[6];
#pragma unroll
    for (int l = 0; l < 6; ++l) w_s[l] = s_wimg + (l < lay.n_layers ? lay.w_off[l] : 0u);

    const int64_t n_items = kShade ? fr.n_pixels : n;
    // tile indices are 32-bit (the host rejects n >= 2^38); only addresses are formed in 64 bits
    const int n_tiles = (int)((n_items + 127) / 128);
    const int n_full = (int)(n_items / 128);                         // tiles [0, n_full) are complete
    const int last_rows = (int)(n_items - (int64_t)n_full * 128);    // live rows of the ragged tile n_full, if any
    const int stride = (int)gridDim.x * NWG;
    const int first = (int)blockIdx.x * NWG + wg;
    auto row_is_live = [&](int tile) { return tile < n_full || (tile == n_full && t < last_rows); };
    uint32_t mma_phase = 0;
    const uint32_t my_stage = s_stage + (uint32_t)wg * T::kStages * T::kStageStride;
    const uint8_t* my_stage_g = g_stage + (size_t)wg * T::kStages * T::kStageStride;
    // per-query frames ride in the same staging buffer when their address allows bulk copies (16-byte aligned)
    const bool frames_bulk = frames != nullptr && (reinterpret_cast<uintptr_t>(frames) & 15u) == 0;

    // eval: full tiles are staged in shared memory by bulk copies, two buffers per warpgroup; the tile processed in
    // iteration k of this warpgroup lives in buffer k & 1 and completes phase (k >> 1) & 1 of that buffer's mbarrier.
    auto tile_is_bulk = [&](int tile) { return !kShade && tile < n_full; };
    auto stage_request = [&](int tile, uint32_t k) {      // one elected lane
        if (tile_is_bulk(tile)) {
            mbar_expect_tx(q_bar + 8u * (k & 1u), T::kStageBytes + (frames_bulk ? T::kFrameBytes : 0u));
            bulk_g2s(my_stage + (k & 1u) * T::kStageStride, q + (int64_t)tile * 128, T::kStageBytes, q_bar + 8u * (k & 1u));
            if (frames_bulk)
                bulk_g2s(my_stage + (k & 1u) * T::kStageStride + T::kStageBytes, frames + (int64_t)tile * 768, T::kFrameBytes,
                         q_bar + 8u * (k & 1u));
        }
    };

    // Hand-over between a warpgroup and its issuer warp, one named barrier (128 arrivals + the 32 waiting issuer lanes):
    // the owning threads never block here.  The MMA that follows is issued only after every owning thread has arrived,
    // which orders both the operand it reads (tcgen05.st ... wait::st) and the accumulator it overwrites
    // (tcgen05.ld ... wait::ld) of all 128 rows before it.
    auto publish = [&]() {
        tmem_wait_st();
        tc_fence_before();
        named_bar_arrive(1 + wg, 160);
    };
    auto await_mma = [&]() {
        mbar_wait(mma_bar, mma_phase);
        mma_phase ^= 1u;
        tc_fence_after();
    };

    // While the grid-dependency wait below blocks (it resolves only when the slowest CTA of the previous kernel has
    // exited: a median of 1.4 us, profiles/r2_eval_timeline.md), pull this CTA's first inputs from HBM into L2.  A
    // prefetch has no destination: data that a predecessor still writes is simply fetched again from L2 after the wait.
    if (issuer && wg < NWG && elect_one()) {
        if constexpr (!kShade) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int tile = first + j * stride;
                if (tile_is_bulk(tile)) {
                    bulk_prefetch_l2(q + (int64_t)tile * 128, T::kStageBytes);
                    if (frames_bulk) bulk_prefetch_l2(frames + (int64_t)tile * 768, T::kFrameBytes);
                }
            }
        } else {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int tile = first + j * stride;
                if (tile < n_full) {
                    bulk_prefetch_l2(fr.pos_fp + (int64_t)tile * 128, 2048u);
                    bulk_prefetch_l2(fr.nrm_u + (int64_t)tile * 128, 2048u);
                    bulk_prefetch_l2(fr.tan_v + (int64_t)tile * 128, 2048u);
                }
            }
        }
        if (wg == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(net.latents) : "memory");
    }
    __syncwarp();

    // ---- everything above touched only this CTA's shared / tensor memory and the immutable weight image; what a
    // previous kernel or copy on the stream may have written (queries, latents) is read from here on ----
    pdl_wait_prior_grid();
    NBSDF_STAMP(tid == 0, net, 2);
    if (!kShade && issuer && wg < NWG) {      // first two query tiles: their HBM latency overlaps the rest of the prologue
        if (elect_one()) {
            stage_request(first, 0u);
            stage_request(first + stride, 1u);
        }
        __syncwarp();
    }
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
    NBSDF_STAMP(tid == 0, net, 3);

    if (issuer) {
        // =========================== MMA / bulk-copy issuer warp of warpgroup wg ===========================
        setmaxnreg_dec<T::kIssuerRegs>();
        // Mirrors the owning warpgroup's static layer sequence: wait for "operand ready", issue the layer, commit.
        // Blocking in tcgen05.mma issue (the tensor pipe's queue is shallow) costs nothing here.
        auto ready = [&]() {
            named_bar_sync(1 + wg, 160);
            tc_fence_after();
        };
        uint32_t k = 0;
        for (int tile = wg < NWG ? first : n_tiles; tile < n_tiles; tile += stride, ++k) {
            ready();
            if (elect_one()) {
                if (k == 0) {
                    stage_request(first + 2 * stride, 2u);    // buffer 0 has been read by every thread of the warpgroup
                    mbar_wait(w_bar, 0);
                    NBSDF_STAMP(wg == 0, net, 4);
                }
                issue_layer<kBf16, T::K1p, H, T::K1p>(acc_d, T::kXDirect ? col0 + T::kXCol : ay_d, one_d, w_s[0], mma_bar);
            }
            __syncwarp();
            ready();
            if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[1], mma_bar);
            __syncwarp();
            if constexpr (T::kMerged) {
                ready();
                if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, col0 + T::kTailCol, w_s[2], mma_bar);
                __syncwarp();
                // the ready() that follows assemble(next) (one round later with kXDirect): staging buffer (k + 1) & 1 is free
                ready();
                if (elect_one()) {
                    issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[3], mma_bar);
                    if (!T::kXDirect) stage_request(tile + 3 * stride, k + 3u);      // after the MMAs: not in the layer chain
                }
                __syncwarp();
                ready();
                if (elect_one()) {
                    issue_layer<kBf16, H + 16, 16, H>(acc_d, ah_d, one_d, w_s[4], mma_bar);
                    if (T::kXDirect) stage_request(tile + 3 * stride, k + 3u);      // after the MMAs: not in the layer chain
                }
                __syncwarp();
            } else {
                ready();
                if (elect_one()) issue_layer<kBf16, H + 16, kFeat, H>(acc_d, ah_d, one_d, w_s[2], mma_bar);
                __syncwarp();
                const int n_rounds = kShade ? lights.n : 1;
                for (int l = 0; l < n_rounds; ++l) {
                    ready();
                    if (elect_one()) issue_layer<kBf16, T::K4p, H, T::K4p>(acc_d, ay_d, one_d, w_s[3], mma_bar);
                    __syncwarp();
                    ready();                                  // eval: follows assemble(next)
                    if (elect_one()) {
                        issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[4], mma_bar);
                        if (!kShade) stage_request(tile + 3 * stride, k + 3u);      // after the MMAs: not in the layer chain
                    }
                    __syncwarp();
                    ready();
                    if (elect_one()) issue_layer<kBf16, H + 16, 16, H>(acc_d, ah_d, one_d, w_s[5], mma_bar);
                    __syncwarp();
                }
            }
        }
    } else {
    // =========================== warpgroup wg: owns rows, runs A1-A4, epilogues, B7, C1-C3 ===========================
    if constexpr (T::kOwnerRegs > T::kBaseRegs) setmaxnreg_inc<T::kOwnerRegs>();

    // shade: this thread's G-buffer texel is requested one tile before it is assembled and lands in registers
    // (52 B/pixel, perfectly coalesced float4 planes)
    float4 pf_pos = make_float4(0.f, 0.f, 0.f, 1.f), pf_nu = make_float4(0.f, 0.f, 1.f, 0.f), pf_tv = make_float4(1.f, 0.f, 0.f, 0.f);
    int pf_mat = -1;
    auto gbuf_request = [&](int tile) {
        const int64_t it = (int64_t)tile * 128 + t;
        pf_pos = make_float4(0.f, 0.f, 0.f, 1.f); pf_nu = make_float4(0.f, 0.f, 1.f, 0.f); pf_tv = make_float4(1.f, 0.f, 0.f, 0.f);
        pf_mat = -1;
        if (row_is_live(tile)) {
            pf_pos = __ldg(fr.pos_fp + it); pf_nu = __ldg(fr.nrm_u + it); pf_tv = __ldg(fr.tan_v + it);
            pf_mat = __ldg(fr.material + it);
        }
    };
    // ---- per-thread state of the tile that starts next (written by assemble(), one tile ahead) ----
    uint32_t x[T::K1p / 2];             // layer-1 operand [z, u', v', lf, c0, c1, c2, 0...] as packed pairs (eval: held in
                                        // registers until the tile starts; shade: stored to TMEM by assemble())
    uint32_t ytail[3];                  // eval: packed [wi, wo]; shade: the same for the light whose MLP-B starts next
    int material = -1;
    float px = 0.0f, py = 0.0f, pz = 0.0f, wo_l[3] = { 0.0f, 0.0f, 1.0f };      // shade: world position, local view direction
    Frame f;                                                                     // shade: local shading frame
#pragma unroll
    for (int c = 0; c < 3; ++c) { f.t[c] = c == 0; f.b[c] = c == 1; f.n[c] = c == 2; }

    // stages A1-A4 for `tile` (iteration k of this warpgroup): fetch + assemble into the state above
    auto assemble = [&](int tile, uint32_t k) {
        const int64_t it = (int64_t)tile * 128 + t;
        float up, vp, lf;
        if constexpr (!kShade) {
            nbsdf_query rec;
            rec.u = rec.v = 0.0f; rec.footprint = 1.0f; rec.material = -1;
            rec.wi[0] = rec.wi[1] = 0.0f; rec.wi[2] = 1.0f; rec.wo[0] = rec.wo[1] = 0.0f; rec.wo[2] = 1.0f;
            const bool bulk = tile_is_bulk(tile);
            const bool direct = !bulk && row_is_live(tile);
            auto unpack = [&](const uint2 w0, const uint2 w1, const uint2 w2, const uint2 w3, const uint2 w4) {
                rec.u = __uint_as_float(w0.x); rec.v = __uint_as_float(w0.y);
                rec.footprint = __uint_as_float(w1.x); rec.material = (int)w1.y;
                rec.wi[0] = __uint_as_float(w2.x); rec.wi[1] = __uint_as_float(w2.y); rec.wi[2] = __uint_as_float(w3.x);
                rec.wo[0] = __uint_as_float(w3.y); rec.wo[1] = __uint_as_float(w4.x); rec.wo[2] = __uint_as_float(w4.y);
            };
            if (bulk) {
                mbar_wait(q_bar + 8u * (k & 1u), (k >> 1) & 1u);
                const uint2* r2 = reinterpret_cast<const uint2*>(my_stage_g + (k & 1u) * T::kStageStride + t * sizeof(nbsdf_query));
                unpack(r2[0], r2[1], r2[2], r2[3], r2[4]);
            } else if (direct) {
                const uint2* r2 = reinterpret_cast<const uint2*>(q + it);
                unpack(__ldg(r2), __ldg(r2 + 1), __ldg(r2 + 2), __ldg(r2 + 3), __ldg(r2 + 4));
            }
            up = wrap01(rec.u); vp = wrap01(rec.v); lf = log_footprint<true>(rec.footprint);
            material = rec.material;
            float wi[3] = { rec.wi[0], rec.wi[1], rec.wi[2] }, wo[3] = { rec.wo[0], rec.wo[1], rec.wo[2] };
            if (frames != nullptr && (bulk || direct)) {
                float2 f0, f1, f2;
                if (bulk && frames_bulk) {
                    const float2* fs = reinterpret_cast<const float2*>(my_stage_g + (k & 1u) * T::kStageStride + T::kStageBytes + t * 24);
                    f0 = fs[0]; f1 = fs[1]; f2 = fs[2];
                } else {
                    const float2* fp2 = reinterpret_cast<const float2*>(frames + 6 * it);
                    f0 = __ldg(fp2); f1 = __ldg(fp2 + 1); f2 = __ldg(fp2 + 2);
                }
                const Frame ff = make_frame(f0.x, f0.y, f1.x, f1.y, f2.x, f2.y);
                to_local(ff, rec.wi[0], rec.wi[1], rec.wi[2], wi);
                to_local(ff, rec.wo[0], rec.wo[1], rec.wo[2], wo);
            }
            ytail[0] = pack2<kBf16, false>(wi[0], wi[1]);
            ytail[1] = pack2<kBf16, false>(wi[2], wo[0]);
            ytail[2] = pack2<kBf16, false>(wo[1], wo[2]);
        } else {
            const float4 pos = pf_pos, nu = pf_nu, tv = pf_tv;
            material = pf_mat;
            gbuf_request(tile + stride);
            px = pos.x; py = pos.y; pz = pos.z;
            f = make_frame(nu.x, nu.y, nu.z, tv.x, tv.y, tv.z);
            const float vx = fr.cam[0] - px, vy = fr.cam[1] - py, vz = fr.cam[2] - pz;
            const float inv = rsqrtf(vx * vx + vy * vy + vz * vz);
            to_local(f, vx * inv, vy * inv, vz * inv, wo_l);
            up = wrap01(nu.w); vp = wrap01(tv.w); lf = log_footprint<true>(pos.w);
        }
        const int m = material < 0 ? 0 : material;
        const uint4* zrow = reinterpret_cast<const uint4*>(g_lat + (size_t)m * L * 2);
#pragma unroll
        for (int i = 0; i < L / 8; ++i) {
            const uint4 z4 = zrow[i];
            x[4 * i] = z4.x; x[4 * i + 1] = z4.y; x[4 * i + 2] = z4.z; x[4 * i + 3] = z4.w;
        }
        x[L / 2] = pack2<kBf16, false>(up, vp);
        x[L / 2 + 1] = pack2<kBf16, false>(lf, tc_bias_const(kBf16, 0));
        x[L / 2 + 2] = pack2<kBf16, false>(tc_bias_const(kBf16, 1), tc_bias_const(kBf16, 2));
#pragma unroll
        for (int i = L / 2 + 3; i < T::K1p / 2; ++i) x[i] = 0u;
        if constexpr (kShade) {         // AY is a region of its own and dead by now (the last layer 4 has completed)
#pragma unroll
            for (int i = 0; i < T::K1p / 2; i += 8) tmem_st8(ay_t + i, x + i);
        }
        if constexpr (T::kXDirect) {    // called after the merged layer has completed: x region and tail block are dead
#pragma unroll
            for (int i = 0; i < T::K1p / 2; i += 8) tmem_st8(lane_taddr + T::kXCol + i, x + i);
            uint32_t y[8] = { ytail[0], ytail[1], ytail[2], c01, c2z, 0u, 0u, 0u };
            tmem_st8(lane_taddr + T::kTailCol, y);
        }
    };

    // shade, stage C1: geometry of light l at this pixel -> packed [wi_local, wo_local] and E * cos
    float w_cur[3] = { 0.0f, 0.0f, 0.0f }, w_nxt[3] = { 0.0f, 0.0f, 0.0f };
    auto light_tail = [&](int l) {
        float wiw[3], E[3], wi[3];
        light_sample(lights.light[l], px, py, pz, wiw, E);
        to_local(f, wiw[0], wiw[1], wiw[2], wi);
        const float cs = fmaxf(wi[2], 0.0f);
        ytail[0] = pack2<kBf16, false>(wi[0], wi[1]);
        ytail[1] = pack2<kBf16, false>(wi[2], wo_l[0]);
        ytail[2] = pack2<kBf16, false>(wo_l[1], wo_l[2]);
#pragma unroll
        for (int c = 0; c < 3; ++c) w_nxt[c] = E[c] * cs;
    };
    // [wi, wo, c0, c1, c2, 0...] -> 8 A-operand columns
    auto store_tail = [&](uint32_t taddr) {
        uint32_t y[8] = { ytail[0], ytail[1], ytail[2], c01, c2z, 0u, 0u, 0u };
        tmem_st8(taddr, y);
    };

    // deferred output of the tile finished last: raw output-layer values, their item and what to do with them
    float o_prev[3] = { 0.0f, 0.0f, 0.0f }, rad[3] = { 0.0f, 0.0f, 0.0f };
    int prev_tile = 0;
    int prev_kind = 0;                  // 0: nothing pending / dead row, 1: store, 2: background (store zeros)
    auto flush_output = [&]() {
        if (prev_kind != 0) {
            float r[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float v = softplus<true>(o_prev[c]);
                r[c] = kShade ? fmaf(v, w_cur[c], rad[c]) : v;
                if (prev_kind == 2) r[c] = 0.0f;
            }
            float* o3 = out + 3 * ((int64_t)prev_tile * 128 + t);
            o3[0] = r[0];
            o3[1] = r[1];
            o3[2] = r[2];
        }
        prev_kind = 0;
        rad[0] = rad[1] = rad[2] = 0.0f;
    };
    auto load_output = [&]() {
        uint32_t o[4];
        tmem_ld4(acc_t, o);
        tmem_wait_ld();
#pragma unroll
        for (int c = 0; c < 3; ++c) o_prev[c] = __uint_as_float(o[c]);
    };

    if (kShade) gbuf_request(first);
    if (first < n_tiles) assemble(first, 0u);

    uint32_t k = 0;
    for (int tile = first; tile < n_tiles; tile += stride, ++k) {
        const int kind = row_is_live(tile) ? (material < 0 ? 2 : 1) : 0;

        // ---- layer-1 operand (and the merged layer's tail block) -> TMEM ----
        if constexpr (!kShade && !T::kXDirect) {
#pragma unroll
            for (int i = 0; i < T::K1p / 2; i += 8) tmem_st8(ay_t + i, x + i);
        }
        if constexpr (T::kMerged && !T::kXDirect) store_tail(lane_taddr + T::kTailCol);

        // ---- MLP-A (B1-B3) ----
        publish();                                        // -> layer 1 (short: nothing is put in its shadow)
        await_mma();
        NBSDF_STAMP(tid == 0 && k == 0, net, 5);
        epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);
        publish();                                        // -> layer 2
        flush_output();                                   // shadow of layer 2: the previous tile's B7 / C2-C3
        NBSDF_STAMP(tid == 0 && k == 1, net, 6);
        if constexpr (kShade) light_tail(0);              //                    and C1 of the first light
        await_mma();
        epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);

        if constexpr (T::kMerged) {
            // ---- merged layers 3+4 (B3-B4): (W4f W3) h2 + W4a [wi, wo] + (W4f b3 + b4); K = H from AH + tail block ----
            publish();                                    // -> merged layer
            if constexpr (!T::kXDirect) assemble(tile + stride, k + 1u);      // shadow of the merged layer: A1-A4 of the next tile
            await_mma();
            epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);
            publish();                                    // -> layer 5
            if constexpr (T::kXDirect) assemble(tile + stride, k + 1u);       // shadow of layer 5 (the merged layer is done)
            await_mma();
            epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);
            publish();                                    // -> layer 6
            await_mma();
            load_output();
        } else {
            publish();                                    // -> layer 3
            await_mma();
            epilogue_to_a<kFeat, false, kBf16>(acc_t, ay_t);      // feat (linear) -> AY columns [0, 16)
            store_tail(ay_t + 16);                                // [wi, wo, c] of the query / of light 0
#pragma unroll
            for (int c = 0; c < 3; ++c) w_cur[c] = kShade ? w_nxt[c] : 1.0f;

            // ---- MLP-B (B4-B7), once per query / once per light (C1-C3) ----
            const int n_rounds = kShade ? lights.n : 1;
            for (int l = 0; l < n_rounds; ++l) {
                publish();                                // -> layer 4 (also: this thread has read the previous light's output)
                if constexpr (kShade) {                   // shadow of layer 4: C2 of the previous light
                    if (l > 0) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            rad[c] = fmaf(softplus<true>(o_prev[c]), w_cur[c], rad[c]);
                            w_cur[c] = w_nxt[c];
                        }
                    }
                } else {
                    assemble(tile + stride, k + 1u);      // shadow of layer 4: A1-A4 of the next tile
                }
                await_mma();
                epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);
                publish();                                // -> layer 5; eval: the issuer also refills the staging buffer just read
                if constexpr (kShade) {                   // shadow of layer 5: C1 of the next light, or A1-A4 of the next tile
                    if (l + 1 < n_rounds) {
                        light_tail(l + 1);
                        store_tail(ay_t + 16);            // layer 4 of light l has completed: its operand may be replaced
                    } else {
                        assemble(tile + stride, k + 1u);
                    }
                }
                await_mma();
                epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);
                publish();                                // -> layer 6
                await_mma();
                load_output();
            }
        }
        prev_tile = tile;
        prev_kind = kind;
    }
    flush_output();
    NBSDF_STAMP(tid == 0, net, 7);
    }   // role

    // ---- teardown ----
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, 512);
    NBSDF_STAMP(tid == 0, net, 8);
}

// ------------------------------------------------------------------------------------------------
template <int L, int H, bool kBf16, bool kShade>
static cudaError_t launch_one(const NetParams& net, int num_sms, const nbsdf_query* q, const float* frames, int64_t n,
                              const FrameParams& fr, const LightParams& lights, float* out, cudaStream_t s, bool init_only)
{
    constexpr int NWG = H == 128 ? 2 : (H == 32 ? (kShade ? 5 : NBSDF_NWG32_EVAL) : (kShade ? NBSDF_NWG64_SHADE : NBSDF_NWG64_EVAL));
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
    cfg.blockDim = dim3(T::kThreads);
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
    // no light: the radiance is exactly zero and the kernel's light loop may assume at least one round
    if (lights.n == 0) return cudaMemsetAsync(out, 0, (size_t)fr.n_pixels * 3 * sizeof(float), s);
    return dispatch<true>(net, precision, num_sms, nullptr, nullptr, 0, fr, lights, out, s, false);
}

}  // namespace nbsdf
