// nbsdf_host.cu -- the C ABI of include/nbsdf.h: context, weight packing, latent table, launches.
// No CPU fallback anywhere: every compute call ends in a kernel launch or an error code.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "nbsdf_common.cuh"

namespace nbsdf {
void pack_fp32(int L, int H, const nbsdf_weights* w, float* blob);
size_t fp32_blob_floats(int L, int H);
size_t encoder_blob_floats(int Fr, int He, int L);
void pack_encoder(int Fr, int He, int L, const nbsdf_encoder_weights* w, float* blob);
cudaError_t launch_encode_latent(const float* w, const float* x_in, int Fr, int He, int L, float* z_row, cudaStream_t s);
}  // namespace nbsdf

using namespace nbsdf;

struct nbsdf_ctx {
    nbsdf_config cfg;
    int num_sms = 0;
    float* d_latents = nullptr;       // [M][L] fp32
    float* d_w32 = nullptr;           // fp32 path blob
    uint8_t* d_wimg_eval = nullptr;   // tensor path shared-memory images (see tc_layout)
    uint8_t* d_wimg_shade = nullptr;
    // Host arrays handed to set_latents / set_albedos are copied into a ring of pinned slots before the call returns;
    // the call blocks only if the ring wraps onto a slot whose copy is still in flight (kRingSlots edits queued).
    static constexpr int kRingSlots = 8;
    float* h_ring = nullptr;          // kRingSlots x ring_slot_floats, pinned
    size_t ring_slot_floats = 0;
    cudaEvent_t ring_ev[kRingSlots] = {};
    bool ring_busy[kRingSlots] = {};
    int ring_next = 0;
    int arch = 0;                     // 0: BASELINE.json decoder (nbsdf_create), 1: paper-structured (nbsdf_create_paper)
    float* d_albedos = nullptr;       // arch 1: [M][12] fp32
    float* d_enc_w = nullptr;         // encoder tail (nbsdf_set_encoder): transposed weights + biases
    float* d_enc_in = nullptr;        // kRingSlots x kEncInFloats: [feature, alpha, beta] of the in-flight encode calls
    int enc_fr = -1, enc_he = 0;
    static constexpr int kEncInFloats = 1024;
    int64_t launches = 0;
    std::string err;
};

static thread_local std::string g_create_err;

// calls that have no context (nbsdf_encode_latent_static) report through nbsdf_last_error(NULL) as nbsdf_create does
namespace nbsdf { void set_global_error(const char* msg) { g_create_err = msg; } }

static int fail(nbsdf_ctx* ctx, int code, const std::string& msg)
{
    if (ctx) ctx->err = msg; else g_create_err = msg;
    return code;
}

static int fail_cuda(nbsdf_ctx* ctx, const char* what, cudaError_t e)
{
    return fail(ctx, NBSDF_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// The library works on ctx->cfg.device; the caller's current device is restored when a call returns.
struct DeviceGuard {
    int prev = -1, dev;
    cudaError_t err;
    explicit DeviceGuard(int d) : dev(d)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    }
    ~DeviceGuard() { if (prev >= 0 && prev != dev) cudaSetDevice(prev); }
};

static cudaError_t ring_create(nbsdf_ctx* ctx, size_t slot_floats)
{
    ctx->ring_slot_floats = slot_floats;
    cudaError_t e = cudaMallocHost(&ctx->h_ring, nbsdf_ctx::kRingSlots * slot_floats * sizeof(float));
    for (int i = 0; e == cudaSuccess && i < nbsdf_ctx::kRingSlots; ++i)
        e = cudaEventCreateWithFlags(&ctx->ring_ev[i], cudaEventDisableTiming);
    return e;
}

// host rows -> next pinned slot -> cudaMemcpyAsync to dst on stream s; never waits unless the ring has wrapped
// The pinned ring cannot live inside a CUDA graph: a captured copy would re-read, on every replay, a slot the host has
// long since reused, and the slot's event would be captured instead of recorded.  Edits go between replays.
static bool stream_is_capturing(cudaStream_t s)
{
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    return cudaStreamIsCapturing(s, &st) == cudaSuccess && st != cudaStreamCaptureStatusNone;
}

static cudaError_t ring_upload(nbsdf_ctx* ctx, float* dst, const float* src_host, size_t n_floats, cudaStream_t s,
                               const float* tail = nullptr, size_t n_tail = 0, float* dst_slots = nullptr, size_t dst_stride = 0,
                               int* slot_out = nullptr)
{
    const int i = ctx->ring_next;
    ctx->ring_next = (i + 1) % nbsdf_ctx::kRingSlots;
    if (ctx->ring_busy[i]) {
        cudaError_t e = cudaEventSynchronize(ctx->ring_ev[i]);
        if (e != cudaSuccess) return e;
        ctx->ring_busy[i] = false;
    }
    float* slot = ctx->h_ring + (size_t)i * ctx->ring_slot_floats;
    if (n_floats) memcpy(slot, src_host, n_floats * sizeof(float));
    if (n_tail) memcpy(slot + n_floats, tail, n_tail * sizeof(float));
    if (dst_slots) dst = dst_slots + (size_t)i * dst_stride;      // one device slot per ring slot
    if (slot_out) *slot_out = i;
    cudaError_t e = cudaMemcpyAsync(dst, slot, (n_floats + n_tail) * sizeof(float), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return e;
    e = cudaEventRecord(ctx->ring_ev[i], s);
    if (e == cudaSuccess) ctx->ring_busy[i] = true;
    return e;
}

// fp32 -> operand type bits, round to nearest even
static uint16_t to_op16(float v, bool bf16)
{
    if (bf16) return __bfloat16_as_ushort(__float2bfloat16_rn(v));
    return __half_as_ushort(__float2half_rn(v));
}

static float from_op16(uint16_t bits, bool bf16)
{
    if (bf16) return __bfloat162float(__ushort_as_bfloat16(bits));
    return __half2float(__ushort_as_half(bits));
}

// Shared-memory image of the tensor path: per layer, per 64-wide K block, N rows of 128 bytes, K-major, with the
// 16-byte chunk index XOR-ed by (row % 8) (the 128-byte swizzle tcgen05 applies when it reads the tile).
// Columns [Kbias, Kbias + 3) of every row hold the three-way 16-bit split of the fp32 bias, each part divided by
// the constant the kernel feeds in that input column (tc_bias_const), so that sum_j w_j * c_j == bias to ~2^-24.
// merged: layers 3 and 4 are multiplied out in double (the feature layer is linear, see tc_layout).
static void pack_tc(int L, int H, bool bf16, bool merged, const nbsdf_weights* w, uint8_t* img)
{
    const TcLayout lay = tc_layout(L, H, merged);
    const int F = kFeat;
    const int Kr6[6] = { L + 3, H, H, F + 6, H, H };
    const int Nr6[6] = { H, H, F, H, H, 3 };
    memset(img, 0, lay.total);
    auto put = [&](int l, int n, int k, uint16_t bits) {
        const int Np = (int)lay.w_rows[l];
        const int kb = k / 64, kk = k % 64;
        const int chunk = (kk / 8) ^ (n % 8);
        const size_t off = lay.w_off[l] + (size_t)kb * Np * 128 + (size_t)n * 128 + (size_t)chunk * 16 + (size_t)(kk % 8) * 2;
        memcpy(img + off, &bits, 2);
    };
    auto put_bias = [&](int l, int n, double b) {
        double r = b;
        for (int j = 0; j < kBiasCols; ++j) {
            const double c = (double)tc_bias_const(bf16, j);
            const uint16_t bits = to_op16((float)(r / c), bf16);
            put(l, n, lay.Kbias[l] + j, bits);
            r -= (double)from_op16(bits, bf16) * c;
        }
    };
    int dst = 0;
    for (int l = 0; l < 6; ++l) {
        if (merged && l == 2) continue;          // folded into layer 4 below
        if (merged && l == 3) {
            for (int n = 0; n < H; ++n) {
                for (int k = 0; k < H; ++k) {
                    double acc = 0.0;
                    for (int j = 0; j < F; ++j) acc += (double)w->W[3][(size_t)n * (F + 6) + j] * (double)w->W[2][(size_t)j * H + k];
                    put(dst, n, k, to_op16((float)acc, bf16));
                }
                for (int i = 0; i < 6; ++i) put(dst, n, H + i, to_op16(w->W[3][(size_t)n * (F + 6) + F + i], bf16));
                double b = (double)w->b[3][n];
                for (int j = 0; j < F; ++j) b += (double)w->W[3][(size_t)n * (F + 6) + j] * (double)w->b[2][j];
                put_bias(dst, n, b);
            }
        } else {
            for (int n = 0; n < Nr6[l]; ++n) {
                for (int k = 0; k < Kr6[l]; ++k) put(dst, n, k, to_op16(w->W[l][(size_t)n * Kr6[l] + k], bf16));
                put_bias(dst, n, (double)w->b[l][n]);
            }
        }
        ++dst;
    }
}

static bool dims_supported(const nbsdf_config* c)
{
    const bool l_ok = c->latent_dim == 8 || c->latent_dim == 16 || c->latent_dim == 32;
    const bool h_ok = c->hidden == 32 || c->hidden == 64 || c->hidden == 128;
    return l_ok && h_ok && c->feat_dim == kFeat && c->max_materials >= 1 && c->max_materials <= 64;
}

extern "C" int nbsdf_create(const nbsdf_config* cfg, const nbsdf_weights* weights, nbsdf_ctx** out)
{
    if (!cfg || !weights || !out) return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create: NULL argument");
    *out = nullptr;
    for (int l = 0; l < 6; ++l)
        if (!weights->W[l] || !weights->b[l]) return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create: NULL weight or bias pointer");
    if (cfg->precision < NBSDF_PREC_FP32 || cfg->precision > NBSDF_PREC_FP16)
        return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create: unknown precision");
    if (!dims_supported(cfg))
        return fail(nullptr, NBSDF_E_UNSUPPORTED,
                    "nbsdf_create: supported dims are latent_dim in {8,16,32}, hidden in {32,64,128}, feat_dim 32, 1..64 materials");
    // bf16 operands are served only where they meet the stated bound (max 1e-2 / mean 2e-3) with margin: the 8-bit
    // significands of the hidden activations put the max at 0.5-1.2e-2 for every H = 32 network and at 1.1e-2 for
    // (L 32, H 64) (tests/quant_emulation.py, no GPU involved) -- rejected, as nbsdf_create_paper does
    if (cfg->precision == NBSDF_PREC_BF16 && (cfg->hidden == 32 || (cfg->latent_dim == 32 && cfg->hidden == 64)))
        return fail(nullptr, NBSDF_E_UNSUPPORTED,
                    "nbsdf_create: bf16 operands cannot meet the 1e-2 max bound at hidden 32 or at (latent_dim 32, hidden 64); "
                    "use NBSDF_PREC_FP16 there");
    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess) return fail_cuda(nullptr, "cudaGetDeviceCount", e);
    if (cfg->device < 0 || cfg->device >= n_dev) return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create: no such device");
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, cfg->device);
    if (e != cudaSuccess) return fail_cuda(nullptr, "cudaGetDeviceProperties", e);
    if (prop.major != 10)
        return fail(nullptr, NBSDF_E_UNSUPPORTED, "nbsdf_create: device is not sm_100 (Blackwell B200); there is no fallback path");
    DeviceGuard guard(cfg->device);
    if (guard.err != cudaSuccess) return fail_cuda(nullptr, "cudaSetDevice", guard.err);

    nbsdf_ctx* ctx = new (std::nothrow) nbsdf_ctx();
    if (!ctx) return fail(nullptr, NBSDF_E_NOMEM, "nbsdf_create: out of host memory");
    ctx->cfg = *cfg;
    ctx->num_sms = prop.multiProcessorCount;
    const int L = cfg->latent_dim, H = cfg->hidden, M = cfg->max_materials;

#define NBSDF_TRY(call, what)                                                    \
    do {                                                                         \
        cudaError_t e_ = (call);                                                 \
        if (e_ != cudaSuccess) {                                                 \
            int rc_ = fail_cuda(nullptr, what, e_);                              \
            nbsdf_destroy(ctx);                                                  \
            return e_ == cudaErrorMemoryAllocation ? NBSDF_E_NOMEM : rc_;        \
        }                                                                        \
    } while (0)

    NBSDF_TRY(cudaMalloc(&ctx->d_latents, (size_t)M * L * sizeof(float)), "cudaMalloc(latents)");
    NBSDF_TRY(cudaMemset(ctx->d_latents, 0, (size_t)M * L * sizeof(float)), "cudaMemset(latents)");
    NBSDF_TRY(ring_create(ctx, (size_t)M * L > nbsdf_ctx::kEncInFloats ? (size_t)M * L : nbsdf_ctx::kEncInFloats), "pinned staging ring");
    if (cfg->precision == NBSDF_PREC_FP32) {
        std::vector<float> blob(fp32_blob_floats(L, H));
        pack_fp32(L, H, weights, blob.data());
        NBSDF_TRY(cudaMalloc(&ctx->d_w32, blob.size() * sizeof(float)), "cudaMalloc(w32)");
        NBSDF_TRY(cudaMemcpy(ctx->d_w32, blob.data(), blob.size() * sizeof(float), cudaMemcpyHostToDevice), "cudaMemcpy(w32)");
        NBSDF_TRY(init_fp32(), "cudaFuncSetAttribute(fp32)");
    } else {
        for (int which = 0; which < 2; ++which) {          // 0: shade image, 1: eval image
            const bool merged = which == 1 && tc_eval_merged(H);
            const TcLayout lay = tc_layout(L, H, merged);
            std::vector<uint8_t> img(lay.total);
            pack_tc(L, H, cfg->precision == NBSDF_PREC_BF16, merged, weights, img.data());
            uint8_t** dst = which ? &ctx->d_wimg_eval : &ctx->d_wimg_shade;
            NBSDF_TRY(cudaMalloc(dst, lay.total), "cudaMalloc(wimg)");
            NBSDF_TRY(cudaMemcpy(*dst, img.data(), lay.total, cudaMemcpyHostToDevice), "cudaMemcpy(wimg)");
        }
        NBSDF_TRY(init_tc(L, H), "cudaFuncSetAttribute(tc)");
    }
#undef NBSDF_TRY
    *out = ctx;
    return NBSDF_OK;
}


// Shared-memory image of the paper-structured decoder: same tile format as pack_tc, seven layers (pd_layout).
static void pack_pd(int H, bool bf16, const nbsdf_paper_weights* w, uint8_t* img)
{
    const PdLayout lay = pd_layout(H);
    const int F = kFeat;
    const int Kr[kPdLayers] = { kPdLatent + kPdBlob, H, F + 5, H, H, H, H };
    const int Nr[kPdLayers] = { H, F, H, H, H, H, 4 };
    memset(img, 0, lay.total);
    for (int l = 0; l < kPdLayers; ++l) {
        const int Np = (int)lay.w_rows[l];
        auto put = [&](int n, int k, uint16_t bits) {
            const int kb = k / 64, kk = k % 64;
            const int chunk = (kk / 8) ^ (n % 8);
            const size_t off = lay.w_off[l] + (size_t)kb * Np * 128 + (size_t)n * 128 + (size_t)chunk * 16 + (size_t)(kk % 8) * 2;
            memcpy(img + off, &bits, 2);
        };
        for (int n = 0; n < Nr[l]; ++n) {
            for (int k = 0; k < Kr[l]; ++k) put(n, k, to_op16(w->W[l][(size_t)n * Kr[l] + k], bf16));
            double r = (double)w->b[l][n];
            for (int j = 0; j < kBiasCols; ++j) {       // three-way 16-bit split of the bias, as in pack_tc
                const double c = (double)tc_bias_const(bf16, j);
                const uint16_t bits = to_op16((float)(r / c), bf16);
                put(n, lay.Kbias[l] + j, bits);
                r -= (double)from_op16(bits, bf16) * c;
            }
        }
    }
}

extern "C" int nbsdf_create_paper(const nbsdf_config* cfg, const nbsdf_paper_weights* weights, nbsdf_ctx** out)
{
    if (!cfg || !weights || !out) return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create_paper: NULL argument");
    *out = nullptr;
    for (int l = 0; l < kPdLayers; ++l)
        if (!weights->W[l] || !weights->b[l]) return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create_paper: NULL weight or bias pointer");
    if (cfg->precision < NBSDF_PREC_FP32 || cfg->precision > NBSDF_PREC_FP16)
        return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create_paper: unknown precision");
    // bf16 operands are rejected, not served at a private tolerance: the log-mapped specular outputs turn the absolute
    // error of 8-bit significands through seven layers into 4e-2 relative, outside the 1e-2 bound
    if (cfg->precision != NBSDF_PREC_FP16 || cfg->latent_dim != kPdLatent || cfg->hidden != 64 || cfg->feat_dim != kFeat ||
        cfg->max_materials < 1 || cfg->max_materials > 64)
        return fail(nullptr, NBSDF_E_UNSUPPORTED,
                    "nbsdf_create_paper: supported are latent_dim 64, hidden 64, feat_dim 32, 1..64 materials, fp16 operands");
    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess) return fail_cuda(nullptr, "cudaGetDeviceCount", e);
    if (cfg->device < 0 || cfg->device >= n_dev) return fail(nullptr, NBSDF_E_INVALID, "nbsdf_create_paper: no such device");
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, cfg->device);
    if (e != cudaSuccess) return fail_cuda(nullptr, "cudaGetDeviceProperties", e);
    if (prop.major != 10)
        return fail(nullptr, NBSDF_E_UNSUPPORTED, "nbsdf_create_paper: device is not sm_100 (Blackwell B200); there is no fallback path");
    DeviceGuard guard(cfg->device);
    if (guard.err != cudaSuccess) return fail_cuda(nullptr, "cudaSetDevice", guard.err);

    nbsdf_ctx* ctx = new (std::nothrow) nbsdf_ctx();
    if (!ctx) return fail(nullptr, NBSDF_E_NOMEM, "nbsdf_create_paper: out of host memory");
    ctx->cfg = *cfg;
    ctx->arch = 1;
    ctx->num_sms = prop.multiProcessorCount;
    const int L = cfg->latent_dim, H = cfg->hidden, M = cfg->max_materials;
#define NBSDF_TRY(call, what)                                                    \
    do {                                                                         \
        cudaError_t e_ = (call);                                                 \
        if (e_ != cudaSuccess) {                                                 \
            int rc_ = fail_cuda(nullptr, what, e_);                              \
            nbsdf_destroy(ctx);                                                  \
            return e_ == cudaErrorMemoryAllocation ? NBSDF_E_NOMEM : rc_;        \
        }                                                                        \
    } while (0)
    NBSDF_TRY(cudaMalloc(&ctx->d_latents, (size_t)M * L * sizeof(float)), "cudaMalloc(latents)");
    NBSDF_TRY(cudaMemset(ctx->d_latents, 0, (size_t)M * L * sizeof(float)), "cudaMemset(latents)");
    NBSDF_TRY(ring_create(ctx, (size_t)M * L > nbsdf_ctx::kEncInFloats ? (size_t)M * L : nbsdf_ctx::kEncInFloats), "pinned staging ring");
    NBSDF_TRY(cudaMalloc(&ctx->d_albedos, (size_t)M * 12 * sizeof(float)), "cudaMalloc(albedos)");
    NBSDF_TRY(cudaMemset(ctx->d_albedos, 0, (size_t)M * 12 * sizeof(float)), "cudaMemset(albedos)");
    {
        const PdLayout lay = pd_layout(H);
        std::vector<uint8_t> img(lay.total);
        pack_pd(H, cfg->precision == NBSDF_PREC_BF16, weights, img.data());
        NBSDF_TRY(cudaMalloc(&ctx->d_wimg_eval, lay.total), "cudaMalloc(wimg)");
        NBSDF_TRY(cudaMemcpy(ctx->d_wimg_eval, img.data(), lay.total, cudaMemcpyHostToDevice), "cudaMemcpy(wimg)");
        ctx->d_wimg_shade = ctx->d_wimg_eval;
    }
    NBSDF_TRY(init_pd(H), "cudaFuncSetAttribute(pd)");
#undef NBSDF_TRY
    *out = ctx;
    return NBSDF_OK;
}

extern "C" int nbsdf_set_albedos(nbsdf_ctx* ctx, int32_t first, int32_t count, const float* albedos_host, void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (ctx->arch != 1) return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_albedos: context was not made by nbsdf_create_paper");
    if (first < 0 || count < 0 || (int64_t)first + count > ctx->cfg.max_materials)
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_albedos: rows out of range");
    if (count == 0) return NBSDF_OK;
    if (!albedos_host) return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_albedos: NULL albedos");
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    if (stream_is_capturing((cudaStream_t)cuda_stream))
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_albedos: the stream is being captured; host edits cannot be part of a CUDA graph "
                                          "(issue them between replays)");
    const cudaError_t e = ring_upload(ctx, ctx->d_albedos + (size_t)first * 12, albedos_host, (size_t)count * 12, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_set_albedos upload", e);
    return NBSDF_OK;
}

extern "C" void nbsdf_destroy(nbsdf_ctx* ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->cfg.device);
    for (int i = 0; i < nbsdf_ctx::kRingSlots; ++i) {
        if (ctx->ring_busy[i] && ctx->ring_ev[i]) cudaEventSynchronize(ctx->ring_ev[i]);
        if (ctx->ring_ev[i]) cudaEventDestroy(ctx->ring_ev[i]);
    }
    if (ctx->h_ring) cudaFreeHost(ctx->h_ring);
    if (ctx->d_enc_w) cudaFree(ctx->d_enc_w);
    if (ctx->d_enc_in) cudaFree(ctx->d_enc_in);
    if (ctx->d_albedos) cudaFree(ctx->d_albedos);
    if (ctx->arch == 1) ctx->d_wimg_shade = nullptr;      // alias of d_wimg_eval
    if (ctx->d_latents) cudaFree(ctx->d_latents);
    if (ctx->d_w32) cudaFree(ctx->d_w32);
    if (ctx->d_wimg_eval) cudaFree(ctx->d_wimg_eval);
    if (ctx->d_wimg_shade) cudaFree(ctx->d_wimg_shade);
    delete ctx;
}

extern "C" const char* nbsdf_last_error(const nbsdf_ctx* ctx)
{
    return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

extern "C" int64_t nbsdf_launch_count(const nbsdf_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int nbsdf_set_latents(nbsdf_ctx* ctx, int32_t first, int32_t count, const float* latents_host, void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (first < 0 || count < 0 || (int64_t)first + count > ctx->cfg.max_materials)
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_latents: rows out of range");
    if (count == 0) return NBSDF_OK;
    if (!latents_host) return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_latents: NULL latents");
    const int L = ctx->cfg.latent_dim;
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    if (stream_is_capturing((cudaStream_t)cuda_stream))
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_latents: the stream is being captured; host edits cannot be part of a CUDA graph "
                                          "(issue them between replays)");
    const cudaError_t e = ring_upload(ctx, ctx->d_latents + (size_t)first * L, latents_host, (size_t)count * L, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_set_latents upload", e);
    return NBSDF_OK;
}

extern "C" int nbsdf_get_latents(nbsdf_ctx* ctx, int32_t first, int32_t count, float* latents_host, void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (first < 0 || count < 0 || (int64_t)first + count > ctx->cfg.max_materials)
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_get_latents: rows out of range");
    if (count == 0) return NBSDF_OK;
    if (!latents_host) return fail(ctx, NBSDF_E_INVALID, "nbsdf_get_latents: NULL latents");
    const int L = ctx->cfg.latent_dim;
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemcpyAsync(latents_host, ctx->d_latents + (size_t)first * L, (size_t)count * L * sizeof(float),
                                    cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_get_latents copy", e);
    return NBSDF_OK;
}

extern "C" int nbsdf_set_encoder(nbsdf_ctx* ctx, const nbsdf_encoder_weights* w)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (!w) return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_encoder: NULL weights");
    for (int l = 0; l < 4; ++l)
        if (!w->W[l] || !w->b[l]) return fail(ctx, NBSDF_E_INVALID, "nbsdf_set_encoder: NULL weight or bias pointer");
    const int Fr = w->feat_width, He = w->hidden, L = ctx->cfg.latent_dim;
    if (!(He == 32 || He == 64 || He == 128 || He == 256) || Fr < 0 || Fr + 2 > nbsdf_ctx::kEncInFloats)
        return fail(ctx, NBSDF_E_UNSUPPORTED, "nbsdf_set_encoder: supported are hidden in {32,64,128,256}, 0 <= feat_width <= 1022");
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    std::vector<float> blob(encoder_blob_floats(Fr, He, L));
    pack_encoder(Fr, He, L, w, blob.data());
    cudaError_t e = cudaDeviceSynchronize();                // an earlier encode call may still read the old weights
    if (e != cudaSuccess) return fail_cuda(ctx, "cudaDeviceSynchronize", e);
    if (ctx->d_enc_w) cudaFree(ctx->d_enc_w);
    ctx->d_enc_w = nullptr;
    ctx->enc_fr = -1;
    e = cudaMalloc(&ctx->d_enc_w, blob.size() * sizeof(float));
    if (e == cudaSuccess && !ctx->d_enc_in)
        e = cudaMalloc(&ctx->d_enc_in, (size_t)nbsdf_ctx::kRingSlots * nbsdf_ctx::kEncInFloats * sizeof(float));
    if (e == cudaSuccess) e = cudaMemcpy(ctx->d_enc_w, blob.data(), blob.size() * sizeof(float), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? fail(ctx, NBSDF_E_NOMEM, "nbsdf_set_encoder: out of device memory")
                                                                 : fail_cuda(ctx, "nbsdf_set_encoder upload", e);
    ctx->enc_fr = Fr;
    ctx->enc_he = He;
    return NBSDF_OK;
}

extern "C" int nbsdf_encode_latent(nbsdf_ctx* ctx, int32_t row, const float* feature_host, float alpha, float beta, void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (ctx->enc_fr < 0) return fail(ctx, NBSDF_E_INVALID, "nbsdf_encode_latent: no encoder installed (nbsdf_set_encoder)");
    if (row < 0 || row >= ctx->cfg.max_materials) return fail(ctx, NBSDF_E_INVALID, "nbsdf_encode_latent: row out of range");
    if (ctx->enc_fr > 0 && !feature_host) return fail(ctx, NBSDF_E_INVALID, "nbsdf_encode_latent: NULL feature");
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    if (stream_is_capturing((cudaStream_t)cuda_stream))
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_encode_latent: the stream is being captured; host edits cannot be part of a CUDA graph "
                                          "(issue them between replays)");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const float ab[2] = { alpha, beta };
    int slot = 0;
    cudaError_t e = ring_upload(ctx, nullptr, feature_host, (size_t)ctx->enc_fr, s, ab, 2, ctx->d_enc_in, nbsdf_ctx::kEncInFloats, &slot);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_encode_latent upload", e);
    const int L = ctx->cfg.latent_dim;
    e = launch_encode_latent(ctx->d_enc_w, ctx->d_enc_in + (size_t)slot * nbsdf_ctx::kEncInFloats, ctx->enc_fr, ctx->enc_he, L,
                             ctx->d_latents + (size_t)row * L, s);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_encode_latent launch", e);
    // the slot (pinned AND device side) is free only when the kernel that reads it has run, not when the copy has:
    // re-record the slot's event behind the launch, so that a wrapped ring waits for the reader even across streams
    e = cudaEventRecord(ctx->ring_ev[slot], s);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_encode_latent event", e);
    ctx->launches += 1;
    return NBSDF_OK;
}

extern "C" int nbsdf_lerp_latents(nbsdf_ctx* ctx, int32_t dst, int32_t a, int32_t b, float t, void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    const int M = ctx->cfg.max_materials;
    if (dst < 0 || dst >= M || a < 0 || a >= M || b < 0 || b >= M)
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_lerp_latents: row out of range");
    if (!(t == t)) return fail(ctx, NBSDF_E_INVALID, "nbsdf_lerp_latents: t is NaN");
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    cudaError_t e = launch_lerp_latents(ctx->d_latents, ctx->cfg.latent_dim, dst, a, b, t, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_lerp_latents launch", e);
    ctx->launches += 1;
    return NBSDF_OK;
}

static NetParams net_params(const nbsdf_ctx* ctx)
{
    NetParams p;
    p.latents = ctx->d_latents;
    p.w32 = ctx->d_w32;
    p.wimg_eval = ctx->d_wimg_eval;
    p.wimg_shade = ctx->d_wimg_shade;
    p.albedos = ctx->d_albedos;
    p.L = ctx->cfg.latent_dim;
    p.H = ctx->cfg.hidden;
    p.M = ctx->cfg.max_materials;
    return p;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

extern "C" int nbsdf_eval(nbsdf_ctx* ctx, const nbsdf_query* q_dev, const float* frames_dev, int64_t n, float* rgb_dev,
                          void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (n < 0) return fail(ctx, NBSDF_E_INVALID, "nbsdf_eval: negative n");
    if (n >= ((int64_t)1 << 37)) return fail(ctx, NBSDF_E_INVALID, "nbsdf_eval: n must be below 2^37 per call");
    if (n == 0) return NBSDF_OK;
    if (!q_dev || !rgb_dev) return fail(ctx, NBSDF_E_INVALID, "nbsdf_eval: NULL buffer");
    if (!aligned16(q_dev) || !aligned16(rgb_dev) || (frames_dev && (reinterpret_cast<uintptr_t>(frames_dev) & 7u)))
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_eval: queries/outputs must be 16-byte aligned, frames 8-byte aligned");
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    cudaError_t e;
    const NetParams net = net_params(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (ctx->arch == 1) e = launch_eval_pd(net, ctx->num_sms, q_dev, frames_dev, n, rgb_dev, s);
    else if (ctx->cfg.precision == NBSDF_PREC_FP32) e = launch_eval_fp32(net, q_dev, frames_dev, n, rgb_dev, s);
    else e = launch_eval_tc(net, ctx->cfg.precision, ctx->num_sms, q_dev, frames_dev, n, rgb_dev, s);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_eval launch", e);
    ctx->launches += 1;
    return NBSDF_OK;
}

extern "C" int nbsdf_shade_frame(nbsdf_ctx* ctx, const nbsdf_gbuffer* g, const nbsdf_light* lights_host, int32_t n_lights,
                                 float* radiance_dev, void* cuda_stream)
{
    if (!ctx) return NBSDF_E_INVALID;
    if (!g) return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: NULL gbuffer");
    if (g->width < 0 || g->height < 0) return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: negative size");
    if (n_lights < 0 || n_lights > NBSDF_MAX_LIGHTS) return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: n_lights must be in [0, 32]");
    if (n_lights > 0 && !lights_host) return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: NULL lights");
    const int64_t npx = (int64_t)g->width * g->height;
    if (npx == 0) return NBSDF_OK;
    if (npx >= ((int64_t)1 << 37)) return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: width * height must be below 2^37");
    if (!g->pos_fp || !g->nrm_u || !g->tan_v || !g->material || !radiance_dev)
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: NULL buffer");
    if (!aligned16(g->pos_fp) || !aligned16(g->nrm_u) || !aligned16(g->tan_v) || !aligned16(radiance_dev) || !aligned16(g->albedo))
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: planes and output must be 16-byte aligned");
    if (g->albedo && ctx->arch != 1)
        return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: an albedo plane needs a context made by nbsdf_create_paper");
    for (int l = 0; l < n_lights; ++l)
        if (lights_host[l].type != 0 && lights_host[l].type != 1)
            return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: light type must be 0 (directional) or 1 (point)");
    DeviceGuard guard(ctx->cfg.device);
    if (guard.err != cudaSuccess) return fail_cuda(ctx, "cudaSetDevice", guard.err);
    cudaError_t e;

    LightParams lp;
    memset(&lp, 0, sizeof lp);
    lp.n = n_lights;
    for (int l = 0; l < n_lights; ++l) {
        lp.light[l] = lights_host[l];
        if (lp.light[l].type == 0) {   // normalise the direction once, in double
            const double x = lp.light[l].vec[0], y = lp.light[l].vec[1], z = lp.light[l].vec[2];
            const double len = sqrt(x * x + y * y + z * z);
            if (!(len > 0.0)) return fail(ctx, NBSDF_E_INVALID, "nbsdf_shade_frame: zero-length light direction");
            lp.light[l].vec[0] = (float)(x / len); lp.light[l].vec[1] = (float)(y / len); lp.light[l].vec[2] = (float)(z / len);
        }
    }
    FrameParams fr;
    fr.pos_fp = reinterpret_cast<const float4*>(g->pos_fp);
    fr.nrm_u = reinterpret_cast<const float4*>(g->nrm_u);
    fr.tan_v = reinterpret_cast<const float4*>(g->tan_v);
    fr.material = g->material;
    fr.albedo = reinterpret_cast<const float4*>(g->albedo);
    fr.n_pixels = npx;
    fr.cam[0] = g->cam_pos[0]; fr.cam[1] = g->cam_pos[1]; fr.cam[2] = g->cam_pos[2];
    const NetParams net = net_params(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (ctx->arch == 1) e = launch_shade_pd(net, ctx->num_sms, fr, lp, radiance_dev, s);
    else if (ctx->cfg.precision == NBSDF_PREC_FP32) e = launch_shade_fp32(net, fr, lp, radiance_dev, s);
    else e = launch_shade_tc(net, ctx->cfg.precision, ctx->num_sms, fr, lp, radiance_dev, s);
    if (e != cudaSuccess) return fail_cuda(ctx, "nbsdf_shade_frame launch", e);
    ctx->launches += 1;
    return NBSDF_OK;
}
