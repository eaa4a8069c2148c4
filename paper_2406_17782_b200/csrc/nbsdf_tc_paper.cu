// nbsdf_tc_paper.cu -- fused tensor-core decoder with the PAPER'S OWN structure (Eq. 8 at 154)
// for sm_100a: latent 64, one-blob encoding 3 -> 24, two fusion layers, five angular-decoder layers with one skip
// connection and leaky ReLU, four log-mapped components combined with the material's albedos.
//
// Same machinery as nbsdf_tc.cu (read its header first): one persistent CTA per SM; NWG warpgroups that each own a
// 128-row tile (thread t <-> row t <-> TMEM lane t) plus one MMA-issuer warp per warpgroup; every layer is a chain of
// tcgen05.mma M = 128 tiles with the activations as A operand in TENSOR MEMORY, the weights resident in shared memory
// and the fp32 accumulator in tensor memory; biases ride inside the contractions; everything that is not a layer runs
// in the shadow of an MMA wait.  What differs:
//   * seven MMA rounds per query (fusion 1-2 once per query / pixel, angular decoder 3-7 once per query / light);
//   * round 1 reads K = 96 from two regions: z (64) from AH and [blob(24), c0, c1, c2] from AY;
//   * the epilogue is a leaky ReLU (fp16 mode: on the packed pair with HMUL2 + HMNMX2; bf16 mode: in fp32) and round 5
//     adds the skip connection from round 3's output, which the owning thread keeps as 32 packed registers;
//   * the output stage inverts the log map of the two specular components and applies Eq. 8.
//
// TMEM columns per warpgroup (H + H/2 + 24):
//   [0, H)              accumulator
//   [H, H + H/2)        AH: z at the start of a tile, then the hidden activations
//   [H + H/2, +24)      AY: [blob(24), c] for round 1 (16 columns), then y = [feat(32), wi(3), wo(2), c] (20 of 24 columns)
#include "nbsdf_common.cuh"
#include "nbsdf_tc_ptx.cuh"

namespace nbsdf {

template <int H, bool kBf16, int NWG, bool kShade>
struct Pd {
    static constexpr PdLayout kLay = pd_layout(H);
    static constexpr int kAccCol = 0;
    static constexpr int kAhCol = H;
    static constexpr int kAyCol = H + H / 2;
    static constexpr int kColsPerWg = H + H / 2 + 24;
    static constexpr int kOneCol = 504;              // CTA-wide constant block (c0, c1, c2, 0...): bias K step of the K = H layers
    static_assert(NWG * kColsPerWg <= kOneCol, "TMEM budget");
    static_assert(H % 64 == 0, "dims");

    static constexpr int kIssuerWarps = (NWG + 3) / 4 * 4;
    static constexpr int kThreads = NWG * 128 + kIssuerWarps * 32;
    static constexpr int kIssuerRegs = 56;
    static constexpr int kBaseRegs = 65536 / kThreads / 8 * 8 > 248 ? 248 : 65536 / kThreads / 8 * 8;
    static constexpr int kOwnerRegsRaw = kBaseRegs + kIssuerWarps * 32 * (kBaseRegs - kIssuerRegs) / (NWG * 128) / 8 * 8;
    static constexpr int kOwnerRegs = kOwnerRegsRaw > 248 ? 248 : kOwnerRegsRaw;
    static_assert(kThreads <= 1024, "CTA size");
    static constexpr bool kTwoLoads = kOwnerRegs >= 136;          // epilogue register budget (see pd_epilogue)

    static constexpr uint32_t kLatRow = kPdLatent * 2 + 16;       // bytes per packed latent row: 16 bytes of padding put
                                                                  // rows of different materials in different banks
    static constexpr uint32_t kLatBytes = 64 * kLatRow;           // packed latent table, max M rows
    static constexpr uint32_t kAlbBytes = 64 * 12 * 4;            // albedo table, max M x 12 fp32
    static constexpr uint32_t kStageBytes = 128 * sizeof(nbsdf_query);      // one tile of query records ...
    static constexpr uint32_t kFrameBytes = 128 * 6 * sizeof(float);         // ... and of per-query frames behind it
    static constexpr uint32_t kStageStride = kStageBytes + kFrameBytes;      // 8192
    static constexpr uint32_t kStages = 2;

    __host__ __device__ static constexpr uint32_t wimg_bytes() { return kLay.total; }
    __host__ __device__ static constexpr uint32_t smem_bytes()
    {
        return 1024u + ((wimg_bytes() + 127u) & ~127u) + kLatBytes + kAlbBytes + NWG * kStages * kStageStride + NWG * 32u + 64u;
    }
};

// leaky ReLU of two accumulator values -> one packed 16-bit pair; kSkip adds the packed pair `skip` first
template <bool kBf16, bool kSkip>
__device__ __forceinline__ uint32_t lrelu_pack(float lo, float hi, uint32_t skip)
{
    if constexpr (kBf16) {
        if constexpr (kSkip) {
            lo += __uint_as_float(skip << 16);
            hi += __uint_as_float(skip & 0xffff0000u);
        }
        lo = fmaxf(lo, kPdSlope * lo);
        hi = fmaxf(hi, kPdSlope * hi);
        return pack2<true, false>(lo, hi);
    } else {
        // on the packed fp16 pair: one FMA-pipe and one ALU-pipe instruction next to the conversion
        uint32_t p = pack2<false, false>(lo, hi);
        __half2 h = *reinterpret_cast<__half2*>(&p);
        if constexpr (kSkip) h = __hadd2(h, *reinterpret_cast<const __half2*>(&skip));
        h = __hmax2(h, __hmul2(h, __float2half2_rn(kPdSlope)));
        return *reinterpret_cast<uint32_t*>(&h);
    }
}

// Epilogue of a hidden layer: acc (N fp32 columns, bias inside) -> leaky ReLU -> packed pairs -> A columns.
// kMode 0: plain; 1: also keep the packed result in skip[] (round 3); 2: add skip[] before the activation (round 5).
template <int N, int kMode, bool kBf16, bool kTwoLoads = false>
__device__ __forceinline__ void pd_epilogue(uint32_t acc_taddr, uint32_t a_taddr, uint32_t (&skip)[32])
{
    if constexpr (kTwoLoads && N == 64) {
        uint32_t v[32], w[32];
        tmem_ld32(acc_taddr, v);
        tmem_ld32(acc_taddr + 32, w);
        tmem_wait_ld();
        uint32_t p[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            p[j] = lrelu_pack<kBf16, kMode == 2>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]), skip[j]);
            if (kMode == 1) skip[j] = p[j];
        }
        tmem_st16(a_taddr, p);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            p[j] = lrelu_pack<kBf16, kMode == 2>(__uint_as_float(w[2 * j]), __uint_as_float(w[2 * j + 1]), skip[16 + j]);
            if (kMode == 1) skip[16 + j] = p[j];
        }
        tmem_st16(a_taddr + 16, p);
        return;
    }
#pragma unroll
    for (int c = 0; c < N; c += 32) {
        uint32_t v[32];
        tmem_ld32(acc_taddr + c, v);
        tmem_wait_ld();
        uint32_t p[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            p[j] = lrelu_pack<kBf16, kMode == 2>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]), skip[(c / 2 + j) & 31]);
            if (kMode == 1) skip[(c / 2 + j) & 31] = p[j];
        }
        tmem_st16(a_taddr + c / 2, p);
    }
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// e^y - 1 for the inverse log map (fast path: ex2 on the special-function unit; series near 0 where it cancels)
__device__ __forceinline__ float fast_expm1(float y)
{
    return fabsf(y) < 0.03f ? y * (1.0f + y * (0.5f + y * 0.16666667f)) : __expf(y) - 1.0f;
}

template <int H, bool kBf16, int NWG, bool kShade>
__global__ void __launch_bounds__(Pd<H, kBf16, NWG, kShade>::kThreads, 1)
pd_kernel(NetParams net, const nbsdf_query* __restrict__ q, const float* __restrict__ frames, int64_t n,
          FrameParams fr, LightParams lights, float* __restrict__ out)
{
    using T = Pd<H, kBf16, NWG, kShade>;
    constexpr int L = kPdLatent;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* gbase = smem_raw + (base - smem_u32(smem_raw));
    constexpr uint32_t kWimgPad = (T::wimg_bytes() + 127u) & ~127u;
    const uint32_t s_wimg = base;
    const uint32_t s_lat = s_wimg + kWimgPad;
    const uint32_t s_alb = s_lat + T::kLatBytes;
    const uint32_t s_stage = s_alb + T::kAlbBytes;
    const uint32_t s_bars = s_stage + NWG * T::kStages * T::kStageStride;
    const uint32_t s_tmem = s_bars + NWG * 32u;
    uint8_t* g_lat = gbase + kWimgPad;
    float* g_alb = reinterpret_cast<float*>(g_lat + T::kLatBytes);
    uint8_t* g_stage = reinterpret_cast<uint8_t*>(g_alb) + T::kAlbBytes;
    uint32_t* g_tmem = reinterpret_cast<uint32_t*>(g_stage + NWG * T::kStages * T::kStageStride + NWG * 32u);

    const int tid = threadIdx.x;
    const int t = tid & 127;               // row within the tile == TMEM lane
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    // warps [0, 4 NWG): the warpgroups that own tile rows; warp 4 NWG + i: the MMA / bulk-copy issuer of warpgroup i
    const bool issuer = warp >= NWG * 4;
    const int wg = issuer ? warp - NWG * 4 : warp >> 2;          // >= NWG: padding warp, idle
    constexpr PdLayout lay = T::kLay;

    // ---- prologue: weight image (before the grid-dependency wait: immutable), latents, albedos, barriers, TMEM ----
    pdl_launch_dependents();
    const uint32_t mma_bar = s_bars + (uint32_t)wg * 32u;
    const uint32_t q_bar = mma_bar + 8u;            // two of them: one per staging buffer
    const uint32_t w_bar = s_tmem + 8u;
    if (warp == 0 && elect_one()) {
        mbar_init(w_bar, 1);
        fence_mbar_init();
        mbar_expect_tx(w_bar, T::wimg_bytes());
        constexpr uint32_t kChunk = 32768u;
        for (uint32_t off = 0; off < T::wimg_bytes(); off += kChunk) {
            const uint32_t bytes = T::wimg_bytes() - off < kChunk ? T::wimg_bytes() - off : kChunk;
            bulk_g2s(s_wimg + off, net.wimg_eval + off, bytes, w_bar);
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
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *g_tmem, 0);
    const uint32_t col0 = tmem_base + (uint32_t)(wg * T::kColsPerWg);                 // lane 0: for MMA operands
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;                      // this warp's lane quarter
    const uint32_t lane_taddr = col0 + lane_off;
    const uint32_t acc_t = lane_taddr + T::kAccCol, ah_t = lane_taddr + T::kAhCol, ay_t = lane_taddr + T::kAyCol;
    const uint32_t acc_d = col0 + T::kAccCol, ah_d = col0 + T::kAhCol, ay_d = col0 + T::kAyCol, one_d = tmem_base + T::kOneCol;

    const uint32_t c01 = pack2<kBf16, false>(tc_bias_const(kBf16, 0), tc_bias_const(kBf16, 1));
    const uint32_t c2z = pack2<kBf16, false>(tc_bias_const(kBf16, 2), 0.0f);
    const uint32_t c12 = pack2<kBf16, false>(tc_bias_const(kBf16, 1), tc_bias_const(kBf16, 2));
    if (!issuer && wg == 0) {
        uint32_t ones[8] = { c01, c2z, 0u, 0u, 0u, 0u, 0u, 0u };
        tmem_st8(tmem_base + lane_off + T::kOneCol, ones);
        tmem_wait_st();
    }
    uint32_t w_s[kPdLayers];
#pragma unroll
    for (int l = 0; l < kPdLayers; ++l) w_s[l] = s_wimg + lay.w_off[l];

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
    const int n_rounds = kShade ? lights.n : 1;

    // eval: full tiles are staged by bulk copies, two buffers per warpgroup (see nbsdf_tc.cu)
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

    // ---- everything above touched only this CTA's shared / tensor memory and the immutable weight image; what a
    // previous kernel or copy on the stream may have written (queries, latents, albedos) is read from here on ----
    pdl_wait_prior_grid();
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
            lat[(i / L) * (T::kLatRow / 2) + (i % L)] =
                kBf16 ? __bfloat16_as_ushort(__float2bfloat16_rn(z)) : __half_as_ushort(__float2half_rn(z));
        }
        for (int i = tid; i < net.M * 12; i += T::kThreads) g_alb[i] = __ldg(net.albedos + i);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    if (issuer) {
        // =========================== MMA / bulk-copy issuer warp of warpgroup wg ===========================
        setmaxnreg_dec<T::kIssuerRegs>();
        auto ready = [&]() {
            named_bar_sync(1 + wg, 160);
            tc_fence_after();
        };
        uint32_t k = 0;
        for (int tile = wg < NWG ? first : n_tiles; tile < n_tiles; tile += stride, ++k) {
            ready();                                              // round 1: z from AH (K 0..63), [blob, c] from AY (K 64..95)
            if (elect_one()) {
                if (k == 0) {
                    stage_request(first + 2 * stride, 2u);        // buffer 0 has been read by every thread of the warpgroup
                    mbar_wait(w_bar, 0);
                }
                issue_layer<kBf16, 96, H, 64>(acc_d, ah_d, ay_d, w_s[0], mma_bar);
            }
            __syncwarp();
            ready();                                              // round 2: fusion layer 2 -> feature
            if (elect_one()) issue_layer<kBf16, H + 16, kFeat, H>(acc_d, ah_d, one_d, w_s[1], mma_bar);
            __syncwarp();
            for (int l = 0; l < n_rounds; ++l) {
                ready();                                          // round 3: y = [feat, wi, wo, c] from AY
                if (elect_one()) issue_layer<kBf16, 48, H, 48>(acc_d, ay_d, one_d, w_s[2], mma_bar);
                __syncwarp();
                ready();
                if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[3], mma_bar);
                __syncwarp();
                ready();                                          // eval: follows assemble(next): staging buffer (k + 1) & 1 is free
                if (elect_one()) {
                    issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[4], mma_bar);
                    if (!kShade) stage_request(tile + 3 * stride, k + 3u);      // after the MMAs: not in the layer chain
                }
                __syncwarp();
                ready();
                if (elect_one()) issue_layer<kBf16, H + 16, H, H>(acc_d, ah_d, one_d, w_s[5], mma_bar);
                __syncwarp();
                ready();
                if (elect_one()) issue_layer<kBf16, H + 16, 16, H>(acc_d, ah_d, one_d, w_s[6], mma_bar);
                __syncwarp();
            }
        }
    } else {
    // =========================== warpgroup wg: owns rows ===========================
    if constexpr (T::kOwnerRegs > T::kBaseRegs) setmaxnreg_inc<T::kOwnerRegs>();

    // shade: G-buffer texel prefetched one tile ahead into registers
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
    int material = -1;
    uint32_t ytail[3] = { 0u, 0u, 0u };   // packed (wi.x, wi.y), (wi.z, wo.x), (wo.y, c0) of the query / of the next light
    float kinv_nxt = 0.01f;               // 1/k of the inverse log map for that query / light: 1/100 above, 1/1000 below the surface
    float px = 0.0f, py = 0.0f, pz = 0.0f, wo_l[2] = { 0.0f, 0.0f };
    Frame f;
#pragma unroll
    for (int c = 0; c < 3; ++c) { f.t[c] = c == 0; f.b[c] = c == 1; f.n[c] = c == 2; }
    const float c0f = tc_bias_const(kBf16, 0);

    auto set_tail = [&](const float wi[3], float wox, float woy) {
        ytail[0] = pack2<kBf16, false>(wi[0], wi[1]);
        ytail[1] = pack2<kBf16, false>(wi[2], wox);
        ytail[2] = pack2<kBf16, false>(woy, c0f);
        kinv_nxt = wi[2] < 0.0f ? 0.001f : 0.01f;
    };
    // [wi, wo.xy, c0, c1, c2, 0...] -> y columns [16, 24)
    auto store_tail = [&]() {
        uint32_t y[8] = { ytail[0], ytail[1], ytail[2], c12, 0u, 0u, 0u, 0u };
        tmem_st8(ay_t + 16, y);
    };

    // Stages A1-A4 for `tile` (iteration k): fetch, wrap, one-blob encode -> AY columns [0, 16) = [blob(24), c0, c1, c2, 0...].
    // Only called when AY is dead: round 3 of the current tile (its last light) has completed.
    auto assemble = [&](int tile, uint32_t k) {
        const int64_t it = (int64_t)tile * 128 + t;
        float up, vp, size;
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
            up = wrap01(rec.u); vp = wrap01(rec.v); size = rec.footprint;
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
            set_tail(wi, wo[0], wo[1]);
        } else {
            const float4 pos = pf_pos, nu = pf_nu, tv = pf_tv;
            material = pf_mat;
            gbuf_request(tile + stride);
            px = pos.x; py = pos.y; pz = pos.z;
            f = make_frame(nu.x, nu.y, nu.z, tv.x, tv.y, tv.z);
            const float vx = fr.cam[0] - px, vy = fr.cam[1] - py, vz = fr.cam[2] - pz;
            const float inv = rsqrtf(vx * vx + vy * vy + vz * vz);
            float wo3[3];
            to_local(f, vx * inv, vy * inv, vz * inv, wo3);
            wo_l[0] = wo3[0]; wo_l[1] = wo3[1];
            up = wrap01(nu.w); vp = wrap01(tv.w); size = pos.w;
        }
        // one-blob: Gaussian of sigma 1/8 centred at s, sampled at the 8 bin centres:
        // exp(-(8 (c_i - s))^2 / 2) = exp2(-log2(e)/2 * (i + 0.5 - 8 s)^2)
        const float s01 = fminf(fmaxf(size, 0.0f), 5.0f) * 0.2f;
        const float sc[3] = { up, vp, s01 };
        uint32_t xb[16];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            // distances pre-scaled by sqrt(log2(e)/2) = 0.84932180: one FFMA, one FMUL, one MUFU.EX2 per channel
            const float s8 = 6.7945744f * sc[a];
#pragma unroll
            for (int i = 0; i < 8; i += 2) {
                const float d0 = ((float)i + 0.5f) * 0.84932180f - s8, d1 = ((float)i + 1.5f) * 0.84932180f - s8;
                xb[a * 4 + i / 2] = pack2<kBf16, false>(ex2_approx(-d0 * d0), ex2_approx(-d1 * d1));
            }
        }
        xb[12] = c01; xb[13] = c2z; xb[14] = 0u; xb[15] = 0u;
        tmem_st16(ay_t, xb);
    };

    // shade, stage C1: geometry of light l -> tail registers, E * |cos| and 1/k
    float w_cur[3] = { 0.0f, 0.0f, 0.0f }, w_nxt[3] = { 0.0f, 0.0f, 0.0f };
    float kinv_cur = 0.01f;
    auto light_tail = [&](int l) {
        float wiw[3], E[3], wi[3];
        light_sample(lights.light[l], px, py, pz, wiw, E);
        to_local(f, wiw[0], wiw[1], wiw[2], wi);
        const float cs = fabsf(wi[2]);
        set_tail(wi, wo_l[0], wo_l[1]);
#pragma unroll
        for (int c = 0; c < 3; ++c) w_nxt[c] = E[c] * cs;
    };

    // output stage: four raw outputs -> components (inverse log map) -> Eq. 8 with the material's albedos
    float o_prev[4] = { 0.0f, 0.0f, 0.0f, 0.0f }, rad[3] = { 0.0f, 0.0f, 0.0f };
    auto bsdf_rgb = [&](int m, float kinv, float rgb[3]) {
        const float4* al = reinterpret_cast<const float4*>(g_alb + 12 * (m < 0 ? 0 : m));
        const float4 a0 = al[0], a1 = al[1], a2 = al[2];            // kd_warp rgb, kd_weft rgb, ks_warp rgb, ks_weft rgb
        const float cw = o_prev[0], cf = o_prev[1];
        const float sw = fast_expm1(o_prev[2]) * kinv, sf = fast_expm1(o_prev[3]) * kinv;
        rgb[0] = a0.x * cw + a0.w * cf + a1.z * sw + a2.y * sf;
        rgb[1] = a0.y * cw + a1.x * cf + a1.w * sw + a2.z * sf;
        rgb[2] = a0.z * cw + a1.y * cf + a2.x * sw + a2.w * sf;
    };
    int prev_tile = 0;
    int prev_kind = 0, prev_mat = 0;    // kind 0: nothing pending / dead row, 1: store, 2: background (store zeros)
    auto flush_output = [&]() {
        if (prev_kind != 0) {
            float r[3];
            bsdf_rgb(prev_mat, kinv_cur, r);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                if (kShade) r[c] = fmaf(r[c], w_cur[c], rad[c]);
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
        for (int c = 0; c < 4; ++c) o_prev[c] = __uint_as_float(o[c]);
    };

    uint32_t skip[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) skip[i] = 0u;

    if (kShade) gbuf_request(first);
    if (first < n_tiles) assemble(first, 0u);

    uint32_t k = 0;
    for (int tile = first; tile < n_tiles; tile += stride, ++k) {
        const int mat_cur = material;
        const int kind = row_is_live(tile) ? (mat_cur < 0 ? 2 : 1) : 0;

        // ---- z -> AH (the previous tile's last layer has completed; [blob, c] is already in AY) ----
        {
            const uint4* zrow = reinterpret_cast<const uint4*>(g_lat + (size_t)(mat_cur < 0 ? 0 : mat_cur) * T::kLatRow);
            uint32_t z[32];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const uint4 z4 = zrow[i];
                z[4 * i] = z4.x; z[4 * i + 1] = z4.y; z[4 * i + 2] = z4.z; z[4 * i + 3] = z4.w;
            }
            tmem_st16(ah_t, z);
            tmem_st16(ah_t + 16, z + 16);
        }
        // ---- fusion ----
        publish();                                        // -> round 1
        await_mma();
        pd_epilogue<H, 0, kBf16, T::kTwoLoads>(acc_t, ah_t, skip);
        publish();                                        // -> round 2
        flush_output();                                   // shadow: the previous tile's output stage
        if constexpr (kShade) light_tail(0);              //         and C1 of the first light
        await_mma();
        pd_epilogue<kFeat, 0, kBf16>(acc_t, ay_t, skip);  // feature -> y columns [0, 16)
        store_tail();
        kinv_cur = kinv_nxt;
#pragma unroll
        for (int c = 0; c < 3; ++c) w_cur[c] = kShade ? w_nxt[c] : 1.0f;

        // ---- angular decoder, once per query / once per light ----
        for (int l = 0; l < n_rounds; ++l) {
            publish();                                    // -> round 3 (also: this thread has read the previous light's output)
            if constexpr (kShade) {                       // shadow: C2 of the previous light
                if (l > 0) {
                    float r[3];
                    bsdf_rgb(mat_cur, kinv_cur, r);
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        rad[c] = fmaf(r[c], w_cur[c], rad[c]);
                        w_cur[c] = w_nxt[c];
                    }
                    kinv_cur = kinv_nxt;
                }
            }
            await_mma();
            pd_epilogue<H, 1, kBf16, T::kTwoLoads>(acc_t, ah_t, skip);  // D1, kept for the skip connection
            publish();                                    // -> round 4
            if constexpr (!kShade) assemble(tile + stride, k + 1u);     // shadow: A1-A4 of the next tile (AY is dead)
            await_mma();
            pd_epilogue<H, 0, kBf16, T::kTwoLoads>(acc_t, ah_t, skip);
            publish();                                    // -> round 5; eval: the issuer also refills the staging buffer just read
            if constexpr (kShade) {                       // shadow: C1 of the next light, or A1-A4 of the next tile
                if (l + 1 < n_rounds) {
                    light_tail(l + 1);
                    store_tail();                         // round 3 of light l has completed: its tail may be replaced
                } else {
                    assemble(tile + stride, k + 1u);
                }
            }
            await_mma();
            pd_epilogue<H, 2, kBf16, T::kTwoLoads>(acc_t, ah_t, skip);  // + skip, then leaky ReLU
            publish();                                    // -> round 6
            await_mma();
            pd_epilogue<H, 0, kBf16, T::kTwoLoads>(acc_t, ah_t, skip);
            publish();                                    // -> round 7
            await_mma();
            load_output();
        }
        prev_tile = tile;
        prev_kind = kind;
        prev_mat = mat_cur;
    }
    flush_output();
    }   // role

    // ---- teardown ----
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, 512);
}

// ------------------------------------------------------------------------------------------------
template <int H, bool kBf16, bool kShade>
static cudaError_t pd_launch_one(const NetParams& net, int num_sms, const nbsdf_query* q, const float* frames, int64_t n,
                                 const FrameParams& fr, const LightParams& lights, float* out, cudaStream_t s, bool init_only)
{
#ifndef NBSDF_PD_NWG_EVAL
#define NBSDF_PD_NWG_EVAL 4
#endif
#ifndef NBSDF_PD_NWG_SHADE
#define NBSDF_PD_NWG_SHADE 3
#endif
    constexpr int NWG = kShade ? NBSDF_PD_NWG_SHADE : NBSDF_PD_NWG_EVAL;
    using T = Pd<H, kBf16, NWG, kShade>;
    auto kern = pd_kernel<H, kBf16, NWG, kShade>;
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
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, net, q, frames, n, fr, lights, out);
}

template <bool kShade>
static cudaError_t pd_dispatch(const NetParams& net, int precision, int num_sms, const nbsdf_query* q, const float* frames,
                               int64_t n, const FrameParams& fr, const LightParams& lights, float* out, cudaStream_t s,
                               bool init_only)
{
    if (net.H != 64) return cudaErrorInvalidValue;
    return precision == NBSDF_PREC_BF16 ? pd_launch_one<64, true, kShade>(net, num_sms, q, frames, n, fr, lights, out, s, init_only)
                                        : pd_launch_one<64, false, kShade>(net, num_sms, q, frames, n, fr, lights, out, s, init_only);
}

cudaError_t init_pd(int H)
{
    NetParams net{};
    net.H = H;
    FrameParams fr{};
    LightParams lt{};
    for (int prec = NBSDF_PREC_BF16; prec <= NBSDF_PREC_FP16; ++prec) {
        cudaError_t e = pd_dispatch<false>(net, prec, 1, nullptr, nullptr, 0, fr, lt, nullptr, 0, true);
        if (e != cudaSuccess) return e;
        e = pd_dispatch<true>(net, prec, 1, nullptr, nullptr, 0, fr, lt, nullptr, 0, true);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_eval_pd(const NetParams& net, int precision, int num_sms, const nbsdf_query* q, const float* frames,
                           int64_t n, float* rgb, cudaStream_t s)
{
    FrameParams fr{};
    LightParams lt{};
    return pd_dispatch<false>(net, precision, num_sms, q, frames, n, fr, lt, rgb, s, false);
}

cudaError_t launch_shade_pd(const NetParams& net, int precision, int num_sms, const FrameParams& fr,
                            const LightParams& lights, float* out, cudaStream_t s)
{
    if (lights.n == 0) return cudaMemsetAsync(out, 0, (size_t)fr.n_pixels * 3 * sizeof(float), s);
    return pd_dispatch<true>(net, precision, num_sms, nullptr, nullptr, 0, fr, lights, out, s, false);
}

}  // namespace nbsdf
