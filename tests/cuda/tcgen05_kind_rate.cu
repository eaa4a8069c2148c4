// tcgen05_kind_rate.cu -- TEST / MEASUREMENT PROGRAM, not product code (throughput half).
//
// PAPER.md:271-273 (sec. 6.5): "other techniques could be used to accelerate its speed further".  The candidate studied in
// BASELINE.md sec. 5 is FP8 (e4m3) operands on the tensor cores.  tests/quant_emulation.py measured what that costs in
// accuracy (8-14x over the bound); this program measures what it would buy ON THE tcgen05 PATH THE KERNELS USE: the
// time of one tcgen05.mma (M = 128, A operand in TMEM, B operand in 128-byte-swizzled shared memory, fp32 accumulator
// in TMEM -- exactly nbsdf_tc.cu's form, same descriptors from nbsdf_tc_ptx.cuh) for kind::f16 (K = 16 per instruction)
// and kind::f8f6f4 with e4m3 operands (K = 32 per instruction), at the decoder's N = 64 and N = 128 tile widths.
// It first CHECKS that the f8f6f4 instruction computes what it should (A = 1, B[n][.] = 1..4 => D[m][n] = K_total * b_n,
// exact in fp32), so that the rate is that of a real e4m3 contraction, then times 4100 back-to-back MMAs on every SM, in
// two issue patterns: n_acc = 1, every instruction accumulates into the SAME tile (the K steps of one layer: a dependent
// chain), and n_acc = 2, alternating between two accumulator tiles (two warpgroups' layers interleaved).
// Prints one JSON line.  Built and run by tests/test_gpu_tcgen05_kind_rate.py (-m gpu).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "nbsdf_tc_ptx.cuh"

using namespace nbsdf;

__device__ __forceinline__ void umma_ts_f8(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

// both operands from shared memory (the form a kernel uses when the A tile is staged by TMA instead of written by an epilogue)
template <bool kF8>
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate)
{
    if (kF8)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
                     ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}

constexpr int kACol = 256;      // A operand: TMEM columns [256, 288) = four K steps of 32 bytes per row
constexpr int kThreads = 128;

// One CTA: D[128][N] = sum over n_mma instructions of A(128 x Kstep) * B(N x Kstep)^T with A = 1 and B[n][.] = b(n).
// out_d (may be NULL): the accumulator, [128][N] fp32.  out_clk[blockIdx.x]: clocks from the first issue to completion.
// kTwoIssuers: lane 0 of warp 0 AND lane 0 of warp 1 each issue n_mma instructions into a tile of their own and commit to
// a barrier of their own (is the per-instruction floor a property of the issuing warp or of the SM's tensor pipe?)
template <bool kF8, int kAcc, bool kASmem = false, bool kTwoIssuers = false>
__global__ void __launch_bounds__(kThreads) rate_kernel(int n_mma, int N, float* out_d, long long* out_clk)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t bar_s, bar2_s;
    __shared__ long long t_s[4];
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5;
    const uint32_t b_s = (smem_u32(smem_raw) + 1023u) & ~1023u;         // N rows of 128 bytes, 1024-byte aligned
    uint8_t* b_g = smem_raw + (b_s - smem_u32(smem_raw));
    // B: every byte / halfword of row n encodes b(n) = (n % 4) + 1, so neither the swizzle nor the K offset matters
    for (int i = tid; i < N * 64; i += kThreads) {
        const int n = i / 64, v = n % 4;
        const uint16_t h16[4] = { 0x3C00, 0x4000, 0x4200, 0x4400 };      // fp16 1, 2, 3, 4
        const uint8_t e4m3[4] = { 0x38, 0x40, 0x44, 0x48 };              // e4m3 1, 2, 3, 4
        reinterpret_cast<uint16_t*>(b_g)[i] = kF8 ? (uint16_t)(e4m3[v] | (e4m3[v] << 8)) : h16[v];
    }
    const uint32_t a_s = b_s + 128u * 128u;                             // kASmem: A tile, 128 rows of 128 bytes, all ones
    if (kASmem)
        for (int i = tid; i < 128 * 32; i += kThreads)
            reinterpret_cast<uint32_t*>(smem_raw + (a_s - smem_u32(smem_raw)))[i] = kF8 ? 0x38383838u : 0x3C003C00u;
    if (warp == 0) { tmem_alloc(smem_u32(&tmem_base_s), 512); tmem_relinquish(); }
    if (tid == 0) { mbar_init(smem_u32(&bar_s), 1); mbar_init(smem_u32(&bar2_s), 1); fence_mbar_init(); }
    fence_proxy_async();                                                // generic-proxy writes of B -> the MMA's async proxy
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;
    const uint32_t lane_t = tmem_base + ((uint32_t)(warp * 32) << 16);
    {   // A = 1 in every element: fp16 pairs 0x3C003C00, e4m3 quads 0x38383838
        uint32_t ones[16];
        for (int j = 0; j < 16; ++j) ones[j] = kF8 ? 0x38383838u : 0x3C003C00u;
        tmem_st16(lane_t + kACol, ones);
        tmem_st16(lane_t + kACol + 16, ones);
        tmem_wait_st();
    }
    tc_fence_before();
    __syncthreads();
    if (tid == 0 || (kTwoIssuers && tid == 32)) {
        const bool second = tid == 32;
        const uint32_t my_bar = smem_u32(second ? &bar2_s : &bar_s);
        tc_fence_after();
        const uint32_t idesc = make_idesc<false>(N);                    // format fields 0: F16 for kind::f16, E4M3 for kind::f8f6f4
        const long long t0 = clock64();
        uint64_t bd[4];
        for (int j = 0; j < 4; ++j) bd[j] = make_b_desc(b_s + (uint32_t)j * 32u);
        const uint32_t a0 = tmem_base + kACol;
        const uint32_t d0 = tmem_base + (second ? (uint32_t)N : 0u);                        // the second issuer owns the tile at column N
        const uint32_t d1 = kAcc == 2 ? tmem_base + (uint32_t)N : d0;
        uint64_t ad[4];
        for (int j = 0; j < 4; ++j) ad[j] = make_b_desc(a_s + (uint32_t)j * 32u);
        auto mma = [&](uint32_t d, int j, uint32_t acc) {
            if (kASmem) umma_ss<kF8>(d, ad[j], bd[j], idesc, acc);
            else if (kF8) umma_ts_f8(d, a0 + (uint32_t)j * 8u, bd[j], idesc, acc);
            else umma_ts(d, a0 + (uint32_t)j * 8u, bd[j], idesc, acc);
        };
        // first group: the accumulate flag is off for the first instruction into each tile (the value check reads this)
        mma(d0, 0, 0u); mma(d1, 1, kAcc == 2 ? 0u : 1u); mma(d0, 2, 1u); mma(d1, 3, 1u);
        // the rest as the kernels issue a layer: operands precomputed, nothing but the instructions in the loop body
        for (int s = 4; s < n_mma; s += 8) {
            mma(d0, 0, 1u); mma(d1, 1, 1u); mma(d0, 2, 1u); mma(d1, 3, 1u);
            mma(d0, 0, 1u); mma(d1, 1, 1u); mma(d0, 2, 1u); mma(d1, 3, 1u);
        }
        umma_commit(my_bar);
        mbar_wait(my_bar, 0);
        const long long t1 = clock64();
        t_s[second ? 2 : 0] = t0; t_s[second ? 3 : 1] = t1;
        if (!kTwoIssuers) out_clk[blockIdx.x] = t1 - t0;
    }
    __syncthreads();
    if (kTwoIssuers && tid == 0) out_clk[blockIdx.x] = (t_s[1] > t_s[3] ? t_s[1] : t_s[3]) - (t_s[0] < t_s[2] ? t_s[0] : t_s[2]);
    tc_fence_after();
    if (out_d != nullptr && blockIdx.x == 0) {
        for (int c0 = 0; c0 < N; c0 += 32) {
            uint32_t r[32];
            tmem_ld32(lane_t + c0, r);
            tmem_wait_ld();
            for (int j = 0; j < 32 && c0 + j < N; ++j) out_d[(size_t)tid * N + c0 + j] = __uint_as_float(r[j]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem_base, 512);
}

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("{\"error\": \"%s at line %d\"}\n", cudaGetErrorString(e_), __LINE__); return 1; } } while (0)

template <bool kF8>
static int run(int N, int n_sms, double clk_per_mma[4], bool* ok)
{
    const size_t smem = (size_t)128 * 128 + 128 * 128 + 1024;          // B (up to 128 rows) | A tile for the smem-A form
    CK(cudaFuncSetAttribute(rate_kernel<kF8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaFuncSetAttribute(rate_kernel<kF8, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaFuncSetAttribute((rate_kernel<kF8, 2, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    CK(cudaFuncSetAttribute((rate_kernel<kF8, 1, false, true>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    float* d_out; long long* d_clk;
    CK(cudaMalloc(&d_out, (size_t)128 * N * sizeof(float)));
    CK(cudaMalloc(&d_clk, (size_t)n_sms * sizeof(long long)));
    // value check: 4 instructions into one accumulator tile, K_total = 4 * (kF8 ? 32 : 16)
    rate_kernel<kF8, 1><<<1, kThreads, smem>>>(4, N, d_out, d_clk);
    CK(cudaDeviceSynchronize());
    std::vector<float> h((size_t)128 * N);
    CK(cudaMemcpy(h.data(), d_out, h.size() * sizeof(float), cudaMemcpyDeviceToHost));
    *ok = true;
    const float kt = 4.0f * (kF8 ? 32.0f : 16.0f);
    for (int m = 0; m < 128; ++m)
        for (int n = 0; n < N; ++n)
            if (h[(size_t)m * N + n] != kt * (float)(n % 4 + 1)) *ok = false;
    // rate: 4100 instructions back to back on every SM, three passes, median CTA of the last pass
    const int n_mma = 4 + 8 * 512;
    std::vector<long long> clk(n_sms);
    for (int n_acc = 1; n_acc <= 4; ++n_acc) {                          // 3: two accumulators, A from shared memory; 4: two issuing warps
        for (int pass = 0; pass < 3; ++pass) {
            if (n_acc == 1) rate_kernel<kF8, 1><<<n_sms, kThreads, smem>>>(n_mma, N, nullptr, d_clk);
            else if (n_acc == 2) rate_kernel<kF8, 2><<<n_sms, kThreads, smem>>>(n_mma, N, nullptr, d_clk);
            else if (n_acc == 3) rate_kernel<kF8, 2, true><<<n_sms, kThreads, smem>>>(n_mma, N, nullptr, d_clk);
            else rate_kernel<kF8, 1, false, true><<<n_sms, kThreads, smem>>>(n_mma, N, nullptr, d_clk);
            CK(cudaDeviceSynchronize());
        }
        CK(cudaMemcpy(clk.data(), d_clk, clk.size() * sizeof(long long), cudaMemcpyDeviceToHost));
        std::sort(clk.begin(), clk.end());
        clk_per_mma[n_acc - 1] = (double)clk[n_sms / 2] / (n_acc == 4 ? 2 * n_mma : n_mma);
    }
    cudaFree(d_out); cudaFree(d_clk);
    return 0;
}

int main()
{
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    if (prop.major != 10) { printf("{\"error\": \"not sm_100\"}\n"); return 1; }
    const int sms = prop.multiProcessorCount;
    const int Ns[4] = { 16, 32, 64, 128 };                // output layer, feature layer, H = 64, H = 128
    double c[2][4][4]; bool ok[2][4];                     // [kind][N][pattern]
    for (int i = 0; i < 4; ++i) {
        if (run<false>(Ns[i], sms, c[0][i], &ok[0][i])) return 1;
        if (run<true>(Ns[i], sms, c[1][i], &ok[1][i])) return 1;
    }
    const char* kind[2] = { "f16", "e4m3" };
    printf("{\"sms\": %d, \"mma_per_pass\": 4100", sms);
    for (int k = 0; k < 2; ++k) {
        printf(", \"%s\": {\"k_per_mma\": %d, \"values_ok\": %s", kind[k], k ? 32 : 16,
               (ok[k][0] && ok[k][1] && ok[k][2] && ok[k][3]) ? "true" : "false");
        for (int i = 0; i < 4; ++i)
            printf(", \"clk_per_mma_n%d_chain\": %.2f, \"clk_per_mma_n%d\": %.2f, \"clk_per_mma_n%d_a_smem\": %.2f, "
                   "\"clk_per_mma_n%d_two_issuers\": %.2f", Ns[i], c[k][i][0], Ns[i], c[k][i][1], Ns[i], c[k][i][2], Ns[i], c[k][i][3]);
        printf("}");
    }
    printf("}\n");
    return 0;
}
