// nbsdf_encoder_static.cu -- nbsdf_encode_latent_static: the encoder tail (the arithmetic of
// nbsdf_encoder.cu) for callers that cannot allocate device memory.
//
// Who that is.  A renderer that handed the whole GPU to its own memory pool at start-up has nothing left for cudaMalloc
// to give, and a frame loop cannot afford the call anyway: cudaMalloc and cudaFree synchronise the device, so an edit
// that allocates stalls every stream for a frame.  nbsdf_set_encoder / nbsdf_encode_latent allocate (weight blob, input
// staging slots, pinned ring).  This entry point allocates nothing, on the device or on the host: weights, feature and
// the output row are the caller's DEVICE buffers, and the only memory of its own that it touches is the fixed array below.
//
// The variant.  One launch per layer instead of one CTA for the whole tail: each output row is one warp's dot product
// over the row-major weights exactly as the caller stores them (no transposed copy to keep), so a layer's rows spread
// over up to 32 CTAs.  The activations that pass from one launch to the next (e0, r, e2) live in g_enc_scratch.
//
// Rules that follow from the scratch being ONE array per GPU, shared by every call of the process on that GPU:
//   * its size is fixed at build time (kScratchFloats * 4 = 3 KB, held by every GPU that loads the library until the
//     process exits); hidden > 256 does not fit and is rejected, as are feat_width > 1022 and latent_dim > 64;
//   * it keeps whatever the previous call left.  Nothing in it has to start at zero: every element a launch reads was
//     written by an earlier launch of the SAME call (e0 by layer 0, r by layer 1, e2 by layer 2), so there is nothing
//     to clear;
//   * two calls whose launches can overlap on the GPU (different streams without an event between them, or two host
//     threads on two streams) race on it and produce garbage.  Calls on one stream are safe: the stream orders them.
//   * the first call on each device looks the array's device address up (cudaGetSymbolAddress: in host code the name
//     `g_enc_scratch` is a host-side handle, NOT a device pointer, and must never be handed to a kernel) and caches it.
//     Make that first call during set-up, before any stream capture.
#include <mutex>

#include "nbsdf_common.cuh"

namespace nbsdf {
void set_global_error(const char* msg);
}

namespace {

constexpr int kMaxHidden = 256, kMaxFeat = 1022, kMaxLatent = 64;
constexpr int kScratchFloats = 3 * kMaxHidden;            // e0 | r | e2
constexpr int kMaxDevices = 64;
constexpr int kWarpsPerCta = 8;
constexpr float kSlope = 0.01f;

static __device__ __align__(256) float g_enc_scratch[kScratchFloats];

std::mutex g_setup_mu;
float* g_scratch_addr[kMaxDevices] = {};                 // device address of g_enc_scratch on device d, once looked up

// out[row] = act(b[row] + W[row] . x (+ skip[row])), one warp per row.  x = in[0 .. n_main) followed by (t0, t1) when
// n_in == n_main + 2 (layer 0: the feature, then alpha and beta, which arrive as kernel arguments).
template <bool kAct>
__global__ void __launch_bounds__(kWarpsPerCta * 32) enc_static_layer(const float* __restrict__ W, const float* __restrict__ b,
                                                                      int n_in, int n_main, int n_out,
                                                                      const float* __restrict__ in, float t0, float t1,
                                                                      const float* __restrict__ skip, float* __restrict__ out)
{
    const int row = blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (row >= n_out) return;
    const float* w = W + (size_t)row * n_in;
    float acc = 0.0f;
    for (int k = lane; k < n_in; k += 32) {
        const float x = k < n_main ? in[k] : (k == n_main ? t0 : t1);
        acc = fmaf(__ldg(w + k), x, acc);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (lane == 0) {
        float v = __ldg(b + row) + acc;
        if (skip != nullptr) v += skip[row];
        out[row] = kAct ? (v >= 0.0f ? v : kSlope * v) : v;
    }
}

int fail(int code, const char* msg)
{
    nbsdf::set_global_error(msg);
    return code;
}

struct Guard {                                           // caller's current device restored on return
    int prev = -1, dev;
    cudaError_t err;
    explicit Guard(int d) : dev(d)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    }
    ~Guard() { if (prev >= 0 && prev != dev) cudaSetDevice(prev); }
};

// With `device` current: the device address of the scratch array there (looked up once per device).
cudaError_t scratch_on_current_device(int device, float** out, bool* wrong_arch)
{
    std::lock_guard<std::mutex> lock(g_setup_mu);
    *wrong_arch = false;
    if (!g_scratch_addr[device]) {
        int major = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
        if (e != cudaSuccess) return e;
        if (major != 10) { *wrong_arch = true; return cudaSuccess; }
        float* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_enc_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[device] = p;
    }
    *out = g_scratch_addr[device];
    return cudaSuccess;
}

}  // namespace

extern "C" int nbsdf_encode_latent_static(int32_t device, const nbsdf_encoder_weights* weights_dev, int32_t latent_dim,
                                          const float* feature_dev, float alpha, float beta, float* z_dev, void* cuda_stream)
{
    if (!weights_dev || !z_dev) return fail(NBSDF_E_INVALID, "nbsdf_encode_latent_static: NULL argument");
    for (int l = 0; l < 4; ++l)
        if (!weights_dev->W[l] || !weights_dev->b[l])
            return fail(NBSDF_E_INVALID, "nbsdf_encode_latent_static: NULL weight or bias pointer");
    const int Fr = weights_dev->feat_width, He = weights_dev->hidden, L = latent_dim;
    if (Fr < 0 || He < 1 || L < 1) return fail(NBSDF_E_INVALID, "nbsdf_encode_latent_static: negative or zero size");
    if (He > kMaxHidden || Fr > kMaxFeat || L > kMaxLatent)
        return fail(NBSDF_E_UNSUPPORTED,
                    "nbsdf_encode_latent_static: the fixed scratch array holds hidden <= 256 (feat_width <= 1022, latent_dim <= 64); "
                    "larger encoders need nbsdf_set_encoder / nbsdf_encode_latent, which allocate");
    if (Fr > 0 && !feature_dev) return fail(NBSDF_E_INVALID, "nbsdf_encode_latent_static: NULL feature");
    if (device < 0 || device >= kMaxDevices) return fail(NBSDF_E_INVALID, "nbsdf_encode_latent_static: no such device");
    Guard guard(device);
    if (guard.err != cudaSuccess) return fail(NBSDF_E_CUDA, "nbsdf_encode_latent_static: cudaSetDevice failed");
    float* scratch = nullptr;
    bool wrong_arch = false;
    cudaError_t e = scratch_on_current_device(device, &scratch, &wrong_arch);
    if (e != cudaSuccess) return fail(NBSDF_E_CUDA, cudaGetErrorString(e));
    if (wrong_arch)
        return fail(NBSDF_E_UNSUPPORTED, "nbsdf_encode_latent_static: device is not sm_100 (Blackwell B200); there is no fallback path");

    float* e0 = scratch;
    float* r = scratch + kMaxHidden;
    float* e2 = scratch + 2 * kMaxHidden;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int threads = kWarpsPerCta * 32;
    const int g_h = (He + kWarpsPerCta - 1) / kWarpsPerCta, g_l = (L + kWarpsPerCta - 1) / kWarpsPerCta;
    const float* const* W = weights_dev->W;
    const float* const* b = weights_dev->b;
    enc_static_layer<true><<<g_h, threads, 0, s>>>(W[0], b[0], Fr + 2, Fr, He, feature_dev, alpha, beta, nullptr, e0);
    enc_static_layer<true><<<g_h, threads, 0, s>>>(W[1], b[1], He, He, He, e0, 0.0f, 0.0f, nullptr, r);
    enc_static_layer<true><<<g_h, threads, 0, s>>>(W[2], b[2], He, He, He, r, 0.0f, 0.0f, e0, e2);   // + e0 before the last leaky ReLU
    enc_static_layer<false><<<g_l, threads, 0, s>>>(W[3], b[3], He, He, L, e2, 0.0f, 0.0f, nullptr, z_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(NBSDF_E_CUDA, cudaGetErrorString(e));
    return NBSDF_OK;
}
