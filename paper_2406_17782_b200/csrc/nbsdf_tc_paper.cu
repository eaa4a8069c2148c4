// nbsdf_tc_paper.cu -- fused tensor-core decoder with the PAPER'S OWN structure (Eq. 8 at 154)
// for sm_100a: latent 64, one-blob encoding 3 -> 24, two fusion layers, five angular-decoder layers with one skip
// connection and leaky ReLU, four log-mapped components combined with the material's albedos.
//
// Same machinery as nbsdf_tc.cu (nbsdf_tc_pipeline.cuh holds what the two share): one persistent CTA per SM; NWG
// warpgroups that each own a 128-row tile (thread t <-> row t <-> TMEM lane t) plus one MMA-issuer warp per warpgroup;
// every layer is a chain of tcgen05.mma M = 128 tiles with the activations as A operand in TENSOR MEMORY, the weights
// resident in shared memory and the fp32 accumulator in tensor memory; biases ride inside the contractions; everything
// that is not a layer runs in the shadow of an MMA wait.  Operands are fp16 (bf16 is rejected at nbsdf_create_paper:
// it cannot meet the tolerance through the log-mapped outputs).  What differs:
//   * seven MMA rounds per query (fusion 1-2 once per query / pixel, angular decoder 3-7 once per query / light);
//   * round 1 reads K = 96 from two regions: z (64) from AH and [blob(24), c0, c1, c2] from AY;
//   * the epilogue is a leaky ReLU (on the packed fp16 pair: HMUL2 + HMNMX2) and round 5
//     adds the skip connection from round 3's output, which the owning thread keeps as 32 packed registers;
//   * the output stage inverts the log map of the two specular components and applies Eq. 8.
//
// TMEM columns per warpgroup (H + H/2 + 24):
//   [0, H)              accumulator
//   [H, H + H/2)        AH: z at the start of a tile, then the hidden activations
//   [H + H/2, +24)      AY: [blob(24), c] for round 1 (16 columns), then y = [feat(32), wi(3), wo(2), c] (20 of 24 columns)
#include <type_traits>

#include "nbsdf_tc_pipeline.cuh"

namespace nbsdf {

constexpr bool kBf16 = false;      // operand type of this kernel: fp16 only (see above)

template <int H, int NWG, bool kShade>
struct Pd {
    using S = PipeShape<NWG>;
    static constexpr PdLayout kLay = pd_layout(H);
    static constexpr int kAccCol = 0;
    static constexpr int kAhCol = H;
    static constexpr int kAyCol = H + H / 2;
    static constexpr int kColsPerWg = H + H / 2 + 24;
    static constexpr int kOneCol = S::kOneCol;
    static_assert(NWG * kColsPerWg <= kOneCol, "TMEM budget");
    static_assert(H % 64 == 0, "dims");
    static constexpr int kThreads = S::kThreads, kOwnerRegs = S::kOwnerRegs, kBaseRegs = S::kBaseRegs, kIssuerRegs = S::kIssuerRegs;
    static constexpr bool kTwoLoads = kOwnerRegs >= 136;          // epilogue register budget (see pd_epilogue)

    static constexpr uint32_t kLatRow = kPdLatent * 2 + 16;       // bytes per packed latent row: 16 bytes of padding put
                                                                  // rows of different materials in different banks
    static constexpr uint32_t kLatBytes = 64 * kLatRow;           // packed latent table, max M rows
    static constexpr uint32_t kAlbBytes = 64 * 12 * 4;            // albedo table, max M x 12 fp32

    __host__ __device__ static constexpr uint32_t wimg_bytes() { return kLay.total; }
    __host__ __device__ static constexpr uint32_t smem_bytes() { return S::smem_bytes(wimg_bytes(), kLatBytes + kAlbBytes); }
};

// leaky ReLU of two accumulator values -> one packed 16-bit pair; kSkip adds the packed pair `skip` first
template <bool kSkip>
__device__ __forceinline__ uint32_t lrelu_pack(float lo, float hi, uint32_t skip)
{
    // on the packed fp16 pair: one FMA-pipe and one ALU-pipe instruction next to the conversion
    uint32_t p = pack2<false, false>(lo, hi);
    __half2 h = *reinterpret_cast<__half2*>(&p);
    if constexpr (kSkip) h = __hadd2(h, *reinterpret_cast<const __half2*>(&skip));
    h = __hmax2(h, __hmul2(h, __float2half2_rn(kPdSlope)));
    return *reinterpret_cast<uint32_t*>(&h);
}

// Epilogue of a hidden layer: acc (N fp32 columns, bias inside) -> leaky ReLU -> packed pairs -> A columns.
// kMode 0: plain; 1: also keep the packed result in skip[] (round 3); 2: add skip[] before the activation (round 5).
template <int N, int kMode, bool kTwoLoads = false>
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
            p[j] = lrelu_pack<kMode == 2>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]), skip[j]);
            if (kMode == 1) skip[j] = p[j];
        }
        tmem_st16(a_taddr, p);
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            p[j] = lrelu_pack<kMode == 2>(__uint_as_float(w[2 * j]), __uint_as_float(w[2 * j + 1]), skip[16 + j]);
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
            p[j] = lrelu_pack<kMode == 2>(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]), skip[(c / 2 + j) & 31]);
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

template <int H, int NWG, bool kShade>
__global__ void __launch_bounds__(Pd<H, NWG, kShade>::kThreads, 1)
pd_kernel(NetParams net, const nbsdf_query* __restrict__ q, const float* __restrict__ frames, int64_t n,
          FrameParams fr, std::conditional_t<kShade, LightParams, NoLightParams> lights, float* __restrict__ out)
{
    using T = Pd<H, NWG, kShade>;
    constexpr int L = kPdLatent;
    extern __shared__ uint8_t smem_raw[];
    constexpr PdLayout lay = T::kLay;

    // ---- prologue (nbsdf_tc_pipeline.cuh), then the latent and albedo tables of this kernel ----
    const uint32_t c01 = pack2<kBf16, false>(tc_bias_const(kBf16, 0), tc_bias_const(kBf16, 1));
    const uint32_t c2z = pack2<kBf16, false>(tc_bias_const(kBf16, 2), 0.0f);
    const uint32_t c12 = pack2<kBf16, false>(tc_bias_const(kBf16, 1), tc_bias_const(kBf16, 2));
    Pipe<NWG, kShade> P;
    P.begin(smem_raw, net.wimg_eval, T::wimg_bytes(), T::kLatBytes + T::kAlbBytes, T::kColsPerWg,
            kShade ? fr.n_pixels : n, q, frames, c01, c2z);
    const int tid = P.tid, t = P.t, wg = P.wg;
    const bool issuer = P.issuer;
    const int n_tiles = P.n_tiles, stride = P.stride, first = P.first;
    const uint32_t col0 = P.col0, lane_taddr = P.lane_taddr, mma_bar = P.mma_bar;
    uint8_t* g_lat = P.g_tables;
    float* g_alb = reinterpret_cast<float*>(g_lat + T::kLatBytes);
    const uint32_t acc_t = lane_taddr + T::kAccCol, ah_t = lane_taddr + T::kAhCol, ay_t = lane_taddr + T::kAyCol;
    const uint32_t acc_d = col0 + T::kAccCol, ah_d = col0 + T::kAhCol, ay_d = col0 + T::kAyCol, one_d = P.tmem_base + T::kOneCol;
    uint32_t w_s[kPdLayers];
#pragma unroll
    for (int l = 0; l < kPdLayers; ++l) w_s[l] = P.s_wimg + lay.w_off[l];
    const int n_rounds = kShade ? lights.n : 1;
    auto row_is_live = [&](int tile) { return P.row_is_live(tile); };
    auto stage_request = [&](int tile, uint32_t k) { P.stage_request(tile, k); };
    auto publish = [&]() { P.publish(); };
    auto await_mma = [&]() { P.await_mma(); };

    P.wait_prior_grid(fr, net.latents);
    {
        uint16_t* lat = reinterpret_cast<uint16_t*>(g_lat);
        for (int i = tid; i < net.M * L; i += T::kThreads)
            lat[(i / L) * (T::kLatRow / 2) + (i % L)] = __half_as_ushort(__float2half_rn(__ldg(net.latents + i)));
        for (int i = tid; i < net.M * 12; i += T::kThreads) g_alb[i] = __ldg(net.albedos + i);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    if (issuer) {
        // =========================== MMA / bulk-copy issuer warp of warpgroup wg ===========================
        setmaxnreg_dec<T::kIssuerRegs>();
        auto ready = [&]() { P.ready(); };
        uint32_t k = 0;
        for (int tile = wg < NWG ? first : n_tiles; tile < n_tiles; tile += stride, ++k) {
            ready();                                              // round 1: z from AH (K 0..63), [blob, c] from AY (K 64..95)
            if (elect_one()) {
                if (k == 0) {
                    stage_request(first + 2 * stride, 2u);        // buffer 0 has been read by every thread of the warpgroup
                    mbar_wait(P.w_bar, 0);
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
    GbufTexel pf;
    pf.clear();
    auto gbuf_request = [&](int tile) { pf.request(fr, (int64_t)tile * 128 + t, row_is_live(tile)); };

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
        float up, vp, size;
        if constexpr (!kShade) {
            nbsdf_query rec;
            float wi[3], wo[3];
            P.fetch_query(tile, k, rec, wi, wo);
            up = wrap01(rec.u); vp = wrap01(rec.v); size = rec.footprint;
            material = rec.material;
            set_tail(wi, wo[0], wo[1]);
        } else {
            const float4 pos = pf.pos, nu = pf.nu, tv = pf.tv;
            material = pf.mat;
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

    // output stage: four raw outputs -> components (inverse log map) -> Eq. 8 with the albedos.
    // Eq. 8 is linear in the components, so the frame kernel accumulates radiance PER COMPONENT over the lights
    // (radc[j][c] = sum_l comp_j E_c |cos|) and applies the albedos once per pixel at the end -- which is also what lets
    // the albedos come from a per-pixel plane (k_d, k_s from albedo maps) at one fetch per pixel.
    float o_prev[4] = { 0.0f, 0.0f, 0.0f, 0.0f };
    float radc[kShade ? 4 : 1][3];
#pragma unroll
    for (int j = 0; j < (kShade ? 4 : 1); ++j) radc[j][0] = radc[j][1] = radc[j][2] = 0.0f;
    auto components = [&](float kinv, float comp[4]) {
        comp[0] = o_prev[0];
        comp[1] = o_prev[1];
        comp[2] = fast_expm1(o_prev[2]) * kinv;
        comp[3] = fast_expm1(o_prev[3]) * kinv;
    };
    auto accumulate = [&](float kinv) {                   // shade: + components of the light just decoded x E |cos|
        float comp[4];
        components(kinv, comp);
#pragma unroll
        for (int j = 0; j < (kShade ? 4 : 1); ++j)
#pragma unroll
            for (int c = 0; c < 3; ++c) radc[j][c] = fmaf(comp[j], w_cur[c], radc[j][c]);
    };
    int prev_tile = 0;
    int prev_kind = 0, prev_mat = 0;    // kind 0: nothing pending / dead row, 1: store, 2: background (store zeros)
    auto flush_output = [&]() {
        if (prev_kind != 0) {
            float4 a0, a1, a2;                            // kd_warp rgb, kd_weft rgb, ks_warp rgb, ks_weft rgb
            if (kShade && fr.albedo != nullptr && prev_kind == 1) {
                const float4* al = fr.albedo + 3 * ((int64_t)prev_tile * 128 + t);
                a0 = __ldg(al); a1 = __ldg(al + 1); a2 = __ldg(al + 2);
            } else {
                const float4* al = reinterpret_cast<const float4*>(g_alb + 12 * (prev_mat < 0 ? 0 : prev_mat));
                a0 = al[0]; a1 = al[1]; a2 = al[2];
            }
            float r[3];
            if constexpr (kShade) {
                accumulate(kinv_cur);                     // the last light
                r[0] = a0.x * radc[0][0] + a0.w * radc[1][0] + a1.z * radc[2][0] + a2.y * radc[3][0];
                r[1] = a0.y * radc[0][1] + a1.x * radc[1][1] + a1.w * radc[2][1] + a2.z * radc[3][1];
                r[2] = a0.z * radc[0][2] + a1.y * radc[1][2] + a2.x * radc[2][2] + a2.w * radc[3][2];
            } else {
                float comp[4];
                components(kinv_cur, comp);
                r[0] = a0.x * comp[0] + a0.w * comp[1] + a1.z * comp[2] + a2.y * comp[3];
                r[1] = a0.y * comp[0] + a1.x * comp[1] + a1.w * comp[2] + a2.z * comp[3];
                r[2] = a0.z * comp[0] + a1.y * comp[1] + a2.x * comp[2] + a2.w * comp[3];
            }
            if (prev_kind == 2) r[0] = r[1] = r[2] = 0.0f;
            P.store_rgb(out, prev_tile, r);
        }
        prev_kind = 0;
#pragma unroll
        for (int j = 0; j < (kShade ? 4 : 1); ++j) radc[j][0] = radc[j][1] = radc[j][2] = 0.0f;
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
        pd_epilogue<H, 0, T::kTwoLoads>(acc_t, ah_t, skip);
        publish();                                        // -> round 2
        flush_output();                                   // shadow: the previous tile's output stage
        if constexpr (kShade) light_tail(0);              //         and C1 of the first light
        await_mma();
        pd_epilogue<kFeat, 0>(acc_t, ay_t, skip);  // feature -> y columns [0, 16)
        store_tail();
        kinv_cur = kinv_nxt;
#pragma unroll
        for (int c = 0; c < 3; ++c) w_cur[c] = kShade ? w_nxt[c] : 1.0f;

        // ---- angular decoder, once per query / once per light ----
        for (int l = 0; l < n_rounds; ++l) {
            publish();                                    // -> round 3 (also: this thread has read the previous light's output)
            if constexpr (kShade) {                       // shadow: C2 of the previous light
                if (l > 0) {
                    accumulate(kinv_cur);
#pragma unroll
                    for (int c = 0; c < 3; ++c) w_cur[c] = w_nxt[c];
                    kinv_cur = kinv_nxt;
                }
            }
            await_mma();
            pd_epilogue<H, 1, T::kTwoLoads>(acc_t, ah_t, skip);  // D1, kept for the skip connection
            publish();                                    // -> round 4
            if constexpr (!kShade) assemble(tile + stride, k + 1u);     // shadow: A1-A4 of the next tile (AY is dead)
            await_mma();
            pd_epilogue<H, 0, T::kTwoLoads>(acc_t, ah_t, skip);
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
            pd_epilogue<H, 2, T::kTwoLoads>(acc_t, ah_t, skip);  // + skip, then leaky ReLU
            publish();                                    // -> round 6
            await_mma();
            pd_epilogue<H, 0, T::kTwoLoads>(acc_t, ah_t, skip);
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

    P.end();
}

// ------------------------------------------------------------------------------------------------
#ifndef NBSDF_PD_NWG_EVAL
#define NBSDF_PD_NWG_EVAL 4
#endif
#ifndef NBSDF_PD_NWG_SHADE
#define NBSDF_PD_NWG_SHADE 3
#endif

template <bool kShade>
static cudaError_t pd_dispatch(const NetParams& net, int num_sms, const nbsdf_query* q, const float* frames, int64_t n,
                               const FrameParams& fr, const LightParams& lights, float* out, cudaStream_t s, bool init_only)
{
    if (net.H != 64) return cudaErrorInvalidValue;
    constexpr int NWG = kShade ? NBSDF_PD_NWG_SHADE : NBSDF_PD_NWG_EVAL;
    using T = Pd<64, NWG, kShade>;
    auto kern = pd_kernel<64, NWG, kShade>;
    if (init_only) return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::smem_bytes());
    if constexpr (kShade) {
        return launch_persistent<NWG>(kern, T::smem_bytes(), num_sms, fr.n_pixels, s, net, q, frames, n, fr, lights, out);
    } else {
        NoLightParams none{};
        return launch_persistent<NWG>(kern, T::smem_bytes(), num_sms, n, s, net, q, frames, n, fr, none, out);
    }
}

cudaError_t init_pd(int H)
{
    NetParams net{};
    net.H = H;
    FrameParams fr{};
    LightParams lt{};
    cudaError_t e = pd_dispatch<false>(net, 1, nullptr, nullptr, 0, fr, lt, nullptr, 0, true);
    if (e != cudaSuccess) return e;
    return pd_dispatch<true>(net, 1, nullptr, nullptr, 0, fr, lt, nullptr, 0, true);
}

cudaError_t launch_eval_pd(const NetParams& net, int num_sms, const nbsdf_query* q, const float* frames, int64_t n, float* rgb,
                           cudaStream_t s)
{
    FrameParams fr{};
    LightParams lt{};
    return pd_dispatch<false>(net, num_sms, q, frames, n, fr, lt, rgb, s, false);
}

cudaError_t launch_shade_pd(const NetParams& net, int num_sms, const FrameParams& fr, const LightParams& lights, float* out,
                            cudaStream_t s)
{
    if (lights.n == 0) return cudaMemsetAsync(out, 0, (size_t)fr.n_pixels * 3 * sizeof(float), s);
    return pd_dispatch<true>(net, num_sms, nullptr, nullptr, 0, fr, lights, out, s, false);
}

}  // namespace nbsdf
