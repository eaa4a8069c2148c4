// nbsdf_tc_pipeline.cuh -- the machinery shared by the two tensor-core kernels (nbsdf_tc.cu: BASELINE.json decoder;
// nbsdf_tc_paper.cu: paper-structured decoder).  What is common to both, and lives here once:
//   * the persistent-CTA skeleton: NWG warpgroups that own 128-row tiles (thread t <-> row t <-> TMEM lane t) plus one
//     MMA / bulk-copy issuer warp per warpgroup; setmaxnreg register hand-over; register budgets;
//   * the shared-memory carve-up (weight image, per-kernel tables, two staging buffers + barriers per warpgroup);
//   * the prologue (weight image by cp.async.bulk BEFORE the grid-dependency wait, mbarrier init, TMEM allocation,
//     the CTA-wide bias-constant block, L2 prefetch of the first tiles under the wait) and the teardown;
//   * tile bookkeeping (32-bit tile indices, ragged tail), the two-buffer bulk-copy staging of query records and
//     per-query frames, the record fetch (stage A1 + A4 for nbsdf_eval), the G-buffer texel prefetch (nbsdf_shade_frame);
//   * the owner <-> issuer hand-over (publish / ready / await_mma) and the launch code.
// What differs per kernel (layer sequence, TMEM column map, epilogues, input encoding, output stage) stays in the .cu.
#pragma once
#include "nbsdf_common.cuh"
#include "nbsdf_tc_ptx.cuh"

namespace nbsdf {

// Threads, registers and staging geometry of a kernel with NWG row-owning warpgroups.
template <int NWG>
struct PipeShape {
    // Warps [0, 4 NWG) own tile rows; then one MMA-issuer warp per warpgroup, padded to whole warpgroups so that
    // setmaxnreg can move the issuers' registers to the row owners.
    static constexpr int kIssuerWarps = (NWG + 3) / 4 * 4;
    static constexpr int kThreads = NWG * 128 + kIssuerWarps * 32;
    static constexpr int kIssuerRegs = 56;
    static constexpr int kBaseRegs = 65536 / kThreads / 8 * 8 > 248 ? 248 : 65536 / kThreads / 8 * 8;      // what ptxas is told
    // only what the issuer warps give back is available to setmaxnreg.inc (not the register file's unallocated rest)
    static constexpr int kOwnerRegsRaw = kBaseRegs + kIssuerWarps * 32 * (kBaseRegs - kIssuerRegs) / (NWG * 128) / 8 * 8;
    static constexpr int kOwnerRegs = kOwnerRegsRaw > 248 ? 248 : kOwnerRegsRaw;
    static_assert(kThreads <= 1024, "CTA size");

    static constexpr uint32_t kStageBytes = 128 * sizeof(nbsdf_query);      // one tile of query records ...
    static constexpr uint32_t kFrameBytes = 128 * 6 * sizeof(float);         // ... and of per-query frames behind it
    static constexpr uint32_t kStageStride = kStageBytes + kFrameBytes;      // 8192
    static constexpr uint32_t kStages = 2;                                   // staging buffers per warpgroup
    static constexpr int kOneCol = 504;      // CTA-wide constant block (c0, c1, c2, 0...): bias K step of the K = H layers

    // dynamic shared memory: [1024-aligned] weight image | tables (per kernel) | staging | barriers | TMEM base + w_bar
    __host__ __device__ static constexpr uint32_t smem_bytes(uint32_t wimg_bytes, uint32_t table_bytes)
    {
        return 1024u + ((wimg_bytes + 127u) & ~127u) + table_bytes + NWG * kStages * kStageStride + NWG * 32u + 64u;
    }
};

// G-buffer texel of one pixel, requested one tile before it is assembled (52 B/pixel, perfectly coalesced planes)
struct GbufTexel {
    float4 pos, nu, tv;
    int mat;
    __device__ __forceinline__ void clear()
    {
        pos = make_float4(0.f, 0.f, 0.f, 1.f); nu = make_float4(0.f, 0.f, 1.f, 0.f); tv = make_float4(1.f, 0.f, 0.f, 0.f);
        mat = -1;
    }
    __device__ __forceinline__ void request(const FrameParams& fr, int64_t it, bool live)
    {
        clear();
        if (live) {
            pos = __ldg(fr.pos_fp + it); nu = __ldg(fr.nrm_u + it); tv = __ldg(fr.tan_v + it);
            mat = __ldg(fr.material + it);
        }
    }
};

// Per-thread view of the pipeline.  Constructed by every thread of the CTA at kernel entry (begin()).
template <int NWG, bool kShade>
struct Pipe {
    using S = PipeShape<NWG>;
    // identity
    int tid, t, warp, wg;
    bool issuer;
    // shared memory (32-bit shared-window addresses for PTX; generic pointers for plain loads)
    uint32_t s_wimg, s_stage, mma_bar, q_bar, w_bar, my_stage;
    uint8_t* g_tables;
    const uint8_t* my_stage_g;
    // tensor memory
    uint32_t tmem_base, col0, lane_off, lane_taddr;
    // tiles: indices are 32-bit; the host rejects n >= 2^37, so that tile + 3 * stride (< 2^30 + 3 * 148 * 6) cannot wrap;
    // only addresses are formed in 64 bits
    int n_tiles, n_full, last_rows, stride, first;
    const nbsdf_query* q;
    const float* frames;
    bool frames_bulk;
    uint32_t mma_phase;

    __device__ __forceinline__ bool row_is_live(int tile) const { return tile < n_full || (tile == n_full && t < last_rows); }
    // eval: full tiles are staged in shared memory by bulk copies, two buffers per warpgroup; the tile processed in
    // iteration k of this warpgroup lives in buffer k & 1 and completes phase (k >> 1) & 1 of that buffer's mbarrier
    __device__ __forceinline__ bool tile_is_bulk(int tile) const { return !kShade && tile >= 0 && tile < n_full; }

    // ---- prologue, part 1: everything that touches only this CTA's shared / tensor memory and the IMMUTABLE weight
    // image, so that with programmatic dependent launch it overlaps the tail of the previous kernel on the stream ----
    __device__ __forceinline__ void begin(uint8_t* smem_raw, const uint8_t* wimg, uint32_t wimg_bytes, uint32_t table_bytes,
                                          int cols_per_wg, int64_t n_items, const nbsdf_query* q_, const float* frames_,
                                          uint32_t c01, uint32_t c2z)
    {
        const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;
        uint8_t* gbase = smem_raw + (base - smem_u32(smem_raw));
        const uint32_t wimg_pad = (wimg_bytes + 127u) & ~127u;
        s_wimg = base;
        g_tables = gbase + wimg_pad;
        s_stage = base + wimg_pad + table_bytes;
        const uint32_t s_bars = s_stage + NWG * S::kStages * S::kStageStride;
        const uint32_t s_tmem = s_bars + NWG * 32u;
        const uint32_t* g_tmem = reinterpret_cast<const uint32_t*>(gbase + (s_tmem - base));

        tid = threadIdx.x;
        t = tid & 127;                                                 // row within the tile == TMEM lane
        warp = __shfl_sync(0xffffffffu, tid >> 5, 0);                  // warp-uniform for the compiler
        issuer = warp >= NWG * 4;                                      // warp 4 NWG + i: issuer of warpgroup i
        wg = issuer ? warp - NWG * 4 : warp >> 2;                      // >= NWG: padding warp, idle
        mma_bar = s_bars + (uint32_t)wg * 32u;
        q_bar = mma_bar + 8u;                                          // two of them: one per staging buffer
        w_bar = s_tmem + 8u;
        mma_phase = 0;

        pdl_launch_dependents();
        if (warp == 0 && elect_one()) {
            mbar_init(w_bar, 1);
            fence_mbar_init();
            // one elected lane streams the whole image in with bulk copies; only the MMA issuers ever wait for it
            mbar_expect_tx(w_bar, wimg_bytes);
            constexpr uint32_t kChunk = 32768u;
            for (uint32_t off = 0; off < wimg_bytes; off += kChunk)
                bulk_g2s(s_wimg + off, wimg + off, wimg_bytes - off < kChunk ? wimg_bytes - off : kChunk, w_bar);
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
        tmem_base = __shfl_sync(0xffffffffu, *g_tmem, 0);
        col0 = tmem_base + (uint32_t)(wg * cols_per_wg);               // lane 0: for MMA operands
        lane_off = (uint32_t)((warp & 3) * 32) << 16;                  // this warp's lane quarter
        lane_taddr = col0 + lane_off;
        if (!issuer && wg == 0) {                                      // the CTA-wide constant block, once per kernel
            uint32_t ones[8] = { c01, c2z, 0u, 0u, 0u, 0u, 0u, 0u };
            tmem_st8(tmem_base + lane_off + S::kOneCol, ones);
            tmem_wait_st();
        }

        n_tiles = (int)((n_items + 127) / 128);
        n_full = (int)(n_items / 128);                                 // tiles [0, n_full) are complete
        last_rows = (int)(n_items - (int64_t)n_full * 128);            // live rows of the ragged tile n_full, if any
        // tile slots in warpgroup-major order (slot = wg * grid + cta): every SM gets the same number of tiles +- 1, and a
        // batch of fewer tiles than slots spreads over all SMs with one warpgroup each instead of filling a few CTAs
        stride = (int)gridDim.x * NWG;
        first = wg * (int)gridDim.x + (int)blockIdx.x;
        q = q_;
        frames = frames_;
        // per-query frames ride in the same staging buffer when their address allows bulk copies (16-byte aligned)
        frames_bulk = frames != nullptr && (reinterpret_cast<uintptr_t>(frames) & 15u) == 0;
        my_stage = s_stage + (uint32_t)wg * S::kStages * S::kStageStride;
        my_stage_g = gbase + (s_stage - base) + (size_t)wg * S::kStages * S::kStageStride;
    }

    // ---- prologue, part 2: wait for the previous kernel / copy on the stream; from here on queries, latents and
    // other tables may be read.  While the wait blocks (it resolves only when the slowest CTA of the previous kernel
    // has exited: a median of 1.4 us, profiles/r2_eval_timeline.md) this CTA's first inputs are pulled from HBM into
    // L2 -- a prefetch has no destination, so data a predecessor still writes is simply fetched again afterwards. ----
    __device__ __forceinline__ void wait_prior_grid(const FrameParams& fr, const void* table0)
    {
        if (issuer && wg < NWG && elect_one()) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int tile = first + j * stride;
                if constexpr (!kShade) {
                    if (tile_is_bulk(tile)) {
                        bulk_prefetch_l2(q + (int64_t)tile * 128, S::kStageBytes);
                        if (frames_bulk) bulk_prefetch_l2(frames + (int64_t)tile * 768, S::kFrameBytes);
                    }
                } else if (tile < n_full) {
                    bulk_prefetch_l2(fr.pos_fp + (int64_t)tile * 128, 2048u);
                    bulk_prefetch_l2(fr.nrm_u + (int64_t)tile * 128, 2048u);
                    bulk_prefetch_l2(fr.tan_v + (int64_t)tile * 128, 2048u);
                }
            }
            if (wg == 0) asm volatile("prefetch.global.L2 [%0];" ::"l"(table0) : "memory");
        }
        __syncwarp();
        pdl_wait_prior_grid();
        if (!kShade && issuer && wg < NWG) {      // first two query tiles: their latency overlaps the table conversion
            if (elect_one()) {
                stage_request(first, 0u);
                stage_request(first + stride, 1u);
            }
            __syncwarp();
        }
    }

    // bulk copy of tile `tile` (iteration k of this warpgroup) into staging buffer k & 1; one elected lane
    __device__ __forceinline__ void stage_request(int tile, uint32_t k) const
    {
        if (tile_is_bulk(tile)) {
            const uint32_t bar = q_bar + 8u * (k & 1u), dst = my_stage + (k & 1u) * S::kStageStride;
            mbar_expect_tx(bar, S::kStageBytes + (frames_bulk ? S::kFrameBytes : 0u));
            bulk_g2s(dst, q + (int64_t)tile * 128, S::kStageBytes, bar);
            if (frames_bulk) bulk_g2s(dst + S::kStageBytes, frames + (int64_t)tile * 768, S::kFrameBytes, bar);
        }
    }

    // Stage A1 (+ A4 when per-query frames are given) of nbsdf_eval for row t of `tile` (iteration k): the query record
    // from the staging buffer (full tiles) or straight from global memory (the ragged tile), directions rotated into
    // the local shading frame.  Dead rows get a harmless default record with material -1.
    __device__ __forceinline__ void fetch_query(int tile, uint32_t k, nbsdf_query& rec, float wi[3], float wo[3]) const
    {
        const int64_t it = (int64_t)tile * 128 + t;
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
        const uint8_t* buf = my_stage_g + (k & 1u) * S::kStageStride;
        if (bulk) {
            mbar_wait(q_bar + 8u * (k & 1u), (k >> 1) & 1u);
            const uint2* r2 = reinterpret_cast<const uint2*>(buf + t * sizeof(nbsdf_query));
            unpack(r2[0], r2[1], r2[2], r2[3], r2[4]);
        } else if (direct) {
            const uint2* r2 = reinterpret_cast<const uint2*>(q + it);
            unpack(__ldg(r2), __ldg(r2 + 1), __ldg(r2 + 2), __ldg(r2 + 3), __ldg(r2 + 4));
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) { wi[c] = rec.wi[c]; wo[c] = rec.wo[c]; }
        if (frames != nullptr && (bulk || direct)) {
            float2 f0, f1, f2;
            if (bulk && frames_bulk) {
                const float2* fs = reinterpret_cast<const float2*>(buf + S::kStageBytes + t * 24);
                f0 = fs[0]; f1 = fs[1]; f2 = fs[2];
            } else {
                const float2* fp2 = reinterpret_cast<const float2*>(frames + 6 * it);
                f0 = __ldg(fp2); f1 = __ldg(fp2 + 1); f2 = __ldg(fp2 + 2);
            }
            const Frame ff = make_frame(f0.x, f0.y, f1.x, f1.y, f2.x, f2.y);
            to_local(ff, rec.wi[0], rec.wi[1], rec.wi[2], wi);
            to_local(ff, rec.wo[0], rec.wo[1], rec.wo[2], wo);
        }
    }

    // ---- hand-over between a warpgroup and its issuer warp: one named barrier (128 arrivals + the 32 waiting issuer
    // lanes); the owning threads never block here.  The MMA that follows is issued only after every owning thread has
    // arrived, which orders both the operand it reads (tcgen05.st ... wait::st) and the accumulator it overwrites
    // (tcgen05.ld ... wait::ld) of all 128 rows before it. ----
    __device__ __forceinline__ void publish() const            // owners: "my part of the next operand is in TMEM"
    {
        tmem_wait_st();
        tc_fence_before();
        named_bar_arrive(1 + wg, 160);
    }
    __device__ __forceinline__ void ready() const              // issuer warp: wait for all 128 owners
    {
        named_bar_sync(1 + wg, 160);
        tc_fence_after();
    }
    // K-split hand-over (a second named barrier per warpgroup): an epilogue that writes its operand in two halves
    // publishes the first half with publish() and the second with publish2(); the issuer issues the K steps that read
    // the first half after ready() and the rest + the commit after ready2(), so the layer's first MMAs run while the
    // owners still convert the second half.  Legal because every owner has READ the whole accumulator (tcgen05.wait::ld)
    // before its first arrive, so the first MMA may overwrite it.
    __device__ __forceinline__ void publish2() const
    {
        tmem_wait_st();
        tc_fence_before();
        named_bar_arrive(1 + NWG + wg, 160);
    }
    __device__ __forceinline__ void ready2() const
    {
        named_bar_sync(1 + NWG + wg, 160);
        tc_fence_after();
    }
    __device__ __forceinline__ void await_mma()                // owners: the layer committed last has completed
    {
        mbar_wait(mma_bar, mma_phase);
        mma_phase ^= 1u;
        tc_fence_after();
    }

    // stage C3 / the store of B7: one RGB triple per row
    __device__ __forceinline__ void store_rgb(float* __restrict__ out, int tile, const float r[3]) const
    {
        float* o3 = out + 3 * ((int64_t)tile * 128 + t);
        o3[0] = r[0];
        o3[1] = r[1];
        o3[2] = r[2];
    }

    __device__ __forceinline__ void end() const
    {
        tc_fence_before();
        __syncthreads();
        if (warp == 0) tmem_dealloc(tmem_base, 512);
    }
};

// One persistent CTA per SM (fewer when there are fewer tiles), programmatic dependent launch allowed so that the
// prologue overlaps the previous kernel's tail.
template <int NWG, typename Kern, typename... Args>
static cudaError_t launch_persistent(Kern kern, uint32_t smem_bytes, int num_sms, int64_t n_items, cudaStream_t s, Args... args)
{
    const int64_t tiles = (n_items + 127) / 128;
    int64_t grid = tiles;                    // one CTA per SM; fewer only when there are fewer tiles than SMs
    if (grid > num_sms) grid = num_sms;
    if (grid < 1) grid = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(PipeShape<NWG>::kThreads);
    cfg.dynamicSmemBytes = smem_bytes;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, args...);
}

}  // namespace nbsdf
