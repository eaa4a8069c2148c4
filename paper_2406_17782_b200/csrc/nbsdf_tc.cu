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

#include <type_traits>

#include "nbsdf_tc_pipeline.cuh"

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
    using S = PipeShape<NWG>;
    static constexpr int kThreads = S::kThreads, kOwnerRegs = S::kOwnerRegs, kBaseRegs = S::kBaseRegs, kIssuerRegs = S::kIssuerRegs;
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
    // K-split hand-over of the K = H layers (Pipe::publish2), where a 64-column epilogue writes its operand in two
    // stores.  Measured (profiles/r2_experiments.md sec. 4): +6 % where x shares the A region (L = 32: the tile starts
    // with a store in its chain), -1.5 % .. -3 % everywhere else (the second barrier costs more than the overlap returns
    // when the chain is already short), so it is enabled only there.
    static constexpr bool kSplit = H == 64 && kMerged && !kXDirect && 2 * NWG + 1 <= 15;
    static constexpr int kColsPerWg = kShade ? H + H / 2 + 24 : H + kAw + (kMerged ? 8 : 0) + (kXDirect ? K1p / 2 : 0);
    static constexpr int kOneCol = S::kOneCol;
    static_assert(NWG * kColsPerWg <= kOneCol, "TMEM budget");
    static_assert(L % 8 == 0 && H % 32 == 0, "dims");
    static_assert(K1p <= 48 && K4p == 48, "x / y hold at most 24 columns");

    // Packed latent table: one 16-bit row per material.  A quarter warp gathers eight rows with one LDS.128 each, which is
    // conflict-free when the eight 16-byte chunks fall into eight different bank groups: the row stride in 16-byte units
    // must be ODD (L = 8: 1; L = 16: 2 + 1 of padding; L = 32: 4 + 1).  Unpadded rows (round 2) put rows m and m + 4
    // (L = 16) or m + 2 (L = 32) on the same banks: material ids sorted vs shuffled measured 37.9 vs 37.2 G queries/s at
    // (L 16, 8 materials) and 34.1 vs 30.3 at (L 32, 64 materials) -- bench.py --case eval_sorted / eval_m64_l32[_sorted].
    static constexpr uint32_t kLatRow = L == 8 ? 16 : L * 2 + 16; // bytes
    static constexpr uint32_t kLatBytes = 64 * (32 * 2 + 16);     // max M x max row

    __host__ __device__ static constexpr uint32_t wimg_bytes() { return kLay.total; }
    __host__ __device__ static constexpr uint32_t smem_bytes() { return S::smem_bytes(wimg_bytes(), kLatBytes); }
};

// Epilogue of a hidden layer: acc (N fp32 columns, bias already inside) -> (ReLU) -> packed 16-bit pairs -> A columns.
// kTwoLoads: 64 columns (two tcgen05.ld) are requested per wait, so the second load's latency hides behind the
// first's; costs 32 more live registers.
struct NoMid { __device__ __forceinline__ void operator()() const {} };

// mid(): called between the two stores of a 64-column epilogue (the K-split hand-over, Pipe::publish2)
template <int N, bool kRelu, bool kBf16, bool kTwoLoads = true, typename Mid = NoMid>
__device__ __forceinline__ void epilogue_to_a(uint32_t acc_taddr, uint32_t a_taddr, Mid mid = Mid())
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
            if (N == 64) mid();
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
            if (N == 64 && c == 32) mid();      // the whole accumulator has been read, the first half is stored
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
          FrameParams fr, std::conditional_t<kShade, LightParams, NoLightParams> lights, float* __restrict__ out)
{
    using T = Tc<L, H, kBf16, NWG, kShade>;
    extern __shared__ uint8_t smem_raw[];
    constexpr TcLayout lay = T::kLay;

    // ---- prologue (nbsdf_tc_pipeline.cuh): weight image, barriers, TMEM, constant block; then the grid-dependency wait
    // with the first tiles prefetched into L2 under it; then the first two query tiles are requested ----
    // bias constants (c0, c1, c2) as packed pairs
    const uint32_t c01 = pack2<kBf16, false>(tc_bias_const(kBf16, 0), tc_bias_const(kBf16, 1));
    const uint32_t c2z = pack2<kBf16, false>(tc_bias_const(kBf16, 2), 0.0f);
    Pipe<NWG, kShade> P;
    P.begin(smem_raw, kShade ? net.wimg_shade : net.wimg_eval, T::wimg_bytes(), T::kLatBytes, T::kColsPerWg,
            kShade ? fr.n_pixels : n, q, frames, c01, c2z);
    const int tid = P.tid, t = P.t, wg = P.wg;
    const bool issuer = P.issuer;
    const int n_tiles = P.n_tiles, stride = P.stride, first = P.first;
    const uint32_t col0 = P.col0, lane_taddr = P.lane_taddr, mma_bar = P.mma_bar;
    uint8_t* g_lat = P.g_tables;
    const uint32_t acc_t = lane_taddr + T::kAccCol, ah_t = lane_taddr + T::kAhCol, ay_t = lane_taddr + T::kAyCol;
    const uint32_t acc_d = col0 + T::kAccCol, ah_d = col0 + T::kAhCol, ay_d = col0 + T::kAyCol, one_d = P.tmem_base + T::kOneCol;
    uint32_t w_s[6];
#pragma unroll
    for (int l = 0; l < 6; ++l) w_s[l] = P.s_wimg + (l < lay.n_layers ? lay.w_off[l] : 0u);
    auto row_is_live = [&](int tile) { return P.row_is_live(tile); };
    auto stage_request = [&](int tile, uint32_t k) { P.stage_request(tile, k); };
    auto publish = [&]() { P.publish(); };
    // epilogue of a 64-wide hidden layer + hand-over of its result as the next layer's operand (K-split where enabled)
    auto epilogue_publish = [&]() {
        if constexpr (T::kSplit) {
            epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t, [&]() { P.publish(); });
            P.publish2();
        } else {
            epilogue_to_a<H, true, kBf16, T::kTwoLoads>(acc_t, ah_t);
            P.publish();
        }
    };
    auto await_mma = [&]() { P.await_mma(); };

    P.wait_prior_grid(fr, net.latents);
    {   // the latent table as 16-bit operand rows
        uint16_t* lat = reinterpret_cast<uint16_t*>(g_lat);
        for (int i = tid; i < net.M * L; i += T::kThreads) {
            const float z = __ldg(net.latents + i);
            lat[(i / L) * (T::kLatRow / 2) + (i % L)] = kBf16 ? __bfloat16_as_ushort(__float2bfloat16_rn(z)) : __half_as_ushort(__float2half_rn(z));
        }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    if (issuer) {
        // =========================== MMA / bulk-copy issuer warp of warpgroup wg ===========================
        setmaxnreg_dec<T::kIssuerRegs>();
        // Mirrors the owning warpgroup's static layer sequence: wait for "operand ready", issue the layer, commit.
        // Blocking in tcgen05.mma issue (the tensor pipe's queue is shallow) costs nothing here.
        auto ready = [&]() { P.ready(); };
        // a K = H layer whose operand arrives in two halves (Pipe::publish2): K steps 0-1 after the first half, the rest
        // (incl. the bias / tail step at address `last`) and the commit after the second
        auto issue_hidden = [&](auto n_tag, uint32_t last, uint32_t w) {
            constexpr int N = decltype(n_tag)::value;
            ready();
            if constexpr (T::kSplit) {
                if (elect_one()) issue_layer<kBf16, H + 16, N, H, 0, 2>(acc_d, ah_d, last, w, mma_bar);
                __syncwarp();
                P.ready2();
                if (elect_one()) issue_layer<kBf16, H + 16, N, H, 2, (H + 16) / 16>(acc_d, ah_d, last, w, mma_bar);
            } else {
                if (elect_one()) issue_layer<kBf16, H + 16, N, H>(acc_d, ah_d, last, w, mma_bar);
            }
        };
        using NH = std::integral_constant<int, H>;
        using N16 = std::integral_constant<int, 16>;
        using NF = std::integral_constant<int, kFeat>;
        uint32_t k = 0;
        for (int tile = wg < NWG ? first : n_tiles; tile < n_tiles; tile += stride, ++k) {
            ready();
            if (elect_one()) {
                if (k == 0) {
                    stage_request(first + 2 * stride, 2u);    // buffer 0 has been read by every thread of the warpgroup
                    mbar_wait(P.w_bar, 0);
                }
                issue_layer<kBf16, T::K1p, H, T::K1p>(acc_d, T::kXDirect ? col0 + T::kXCol : ay_d, one_d, w_s[0], mma_bar);
            }
            __syncwarp();
            issue_hidden(NH{}, one_d, w_s[1]);
            __syncwarp();
            if constexpr (T::kMerged) {
                issue_hidden(NH{}, col0 + T::kTailCol, w_s[2]);
                __syncwarp();
                // the ready() that follows assemble(next) (one round later with kXDirect): staging buffer (k + 1) & 1 is free
                issue_hidden(NH{}, one_d, w_s[3]);
                if (!T::kXDirect && elect_one()) stage_request(tile + 3 * stride, k + 3u);      // after the MMAs: not in the layer chain
                __syncwarp();
                issue_hidden(N16{}, one_d, w_s[4]);
                if (T::kXDirect && elect_one()) stage_request(tile + 3 * stride, k + 3u);       // after the MMAs: not in the layer chain
                __syncwarp();
            } else {
                issue_hidden(NF{}, one_d, w_s[2]);
                __syncwarp();
                const int n_rounds = kShade ? lights.n : 1;
                for (int l = 0; l < n_rounds; ++l) {
                    ready();
                    if (elect_one()) issue_layer<kBf16, T::K4p, H, T::K4p>(acc_d, ay_d, one_d, w_s[3], mma_bar);
                    __syncwarp();
                    issue_hidden(NH{}, one_d, w_s[4]);        // eval: follows assemble(next)
                    if (!kShade && elect_one()) stage_request(tile + 3 * stride, k + 3u);      // after the MMAs: not in the layer chain
                    __syncwarp();
                    issue_hidden(N16{}, one_d, w_s[5]);
                    __syncwarp();
                }
            }
        }
    } else {
    // =========================== warpgroup wg: owns rows, runs A1-A4, epilogues, B7, C1-C3 ===========================
    if constexpr (T::kOwnerRegs > T::kBaseRegs) setmaxnreg_inc<T::kOwnerRegs>();

    // shade: this thread's G-buffer texel is requested one tile before it is assembled and lands in registers
    // (52 B/pixel, perfectly coalesced float4 planes)
    GbufTexel pf;
    pf.clear();
    auto gbuf_request = [&](int tile) { pf.request(fr, (int64_t)tile * 128 + t, row_is_live(tile)); };
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
        float up, vp, lf;
        if constexpr (!kShade) {
            nbsdf_query rec;
            float wi[3], wo[3];
            P.fetch_query(tile, k, rec, wi, wo);
            up = wrap01(rec.u); vp = wrap01(rec.v); lf = log_footprint<true>(rec.footprint);
            material = rec.material;
            ytail[0] = pack2<kBf16, false>(wi[0], wi[1]);
            ytail[1] = pack2<kBf16, false>(wi[2], wo[0]);
            ytail[2] = pack2<kBf16, false>(wo[1], wo[2]);
        } else {
            const float4 pos = pf.pos, nu = pf.nu, tv = pf.tv;
            material = pf.mat;
            gbuf_request(tile + stride);
            px = pos.x; py = pos.y; pz = pos.z;
            f = make_frame(nu.x, nu.y, nu.z, tv.x, tv.y, tv.z);
            const float vx = fr.cam[0] - px, vy = fr.cam[1] - py, vz = fr.cam[2] - pz;
            const float inv = rsqrtf(vx * vx + vy * vy + vz * vz);
            to_local(f, vx * inv, vy * inv, vz * inv, wo_l);
            up = wrap01(nu.w); vp = wrap01(tv.w); lf = log_footprint<true>(pos.w);
        }
        const int m = material < 0 ? 0 : material;
        const uint4* zrow = reinterpret_cast<const uint4*>(g_lat + (size_t)m * T::kLatRow);
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
            P.store_rgb(out, prev_tile, r);
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
        epilogue_publish();                               // -> layer 2
        flush_output();                                   // shadow of layer 2: the previous tile's B7 / C2-C3
        if constexpr (kShade) light_tail(0);              //                    and C1 of the first light
        await_mma();
        epilogue_publish();                               // -> merged layer / layer 3

        if constexpr (T::kMerged) {
            // ---- merged layers 3+4 (B3-B4): (W4f W3) h2 + W4a [wi, wo] + (W4f b3 + b4); K = H from AH + tail block ----
            if constexpr (!T::kXDirect) assemble(tile + stride, k + 1u);      // shadow of the merged layer: A1-A4 of the next tile
            await_mma();
            epilogue_publish();                           // -> layer 5
            if constexpr (T::kXDirect) assemble(tile + stride, k + 1u);       // shadow of layer 5 (the merged layer is done)
            await_mma();
            epilogue_publish();                           // -> layer 6
            await_mma();
            load_output();
        } else {
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
                epilogue_publish();                       // -> layer 5; eval: the issuer also refills the staging buffer just read
                if constexpr (kShade) {                   // shadow of layer 5: C1 of the next light, or A1-A4 of the next tile
                    if (l + 1 < n_rounds) {
                        light_tail(l + 1);
                        store_tail(ay_t + 16);            // layer 4 of light l has completed: its operand may be replaced
                    } else {
                        assemble(tile + stride, k + 1u);
                    }
                }
                await_mma();
                epilogue_publish();                       // -> layer 6
                await_mma();
                load_output();
            }
        }
        prev_tile = tile;
        prev_kind = kind;
    }
    flush_output();
    }   // role

    P.end();
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
    if constexpr (kShade) {
        return launch_persistent<NWG>(kern, T::smem_bytes(), num_sms, fr.n_pixels, s, net, q, frames, n, fr, lights, out);
    } else {
        NoLightParams none{};
        return launch_persistent<NWG>(kern, T::smem_bytes(), num_sms, n, s, net, q, frames, n, fr, none, out);
    }
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
