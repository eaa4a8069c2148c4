// nbsdf_encoder.cu -- the encoder tail on the device:
//   x = [feature(Fr), alpha, beta] -> e0 = lrelu(E0 x + b0) -> r = lrelu(E1 e0 + b1) -> e2 = lrelu(E2 r + b2 + e0)
//   -> z = E3 e2 + b3, written straight into row `row` of the context's latent table on the caller's stream, so that
// "infer the encoder to update the material latent vector" is one small kernel and no host round trip.
// Batch 1, ~0.3 MB of weights: latency-bound by construction, so ONE CTA, fp32 FMA, weights stored transposed
// ([k][n_out]: consecutive threads read consecutive addresses), K split over 256 / n_out thread groups whose partial
// sums are added in group order.  The ResNet-18 trunk that produces `feature` is out of scope (no textures, no weights).
#include "nbsdf_common.cuh"

namespace nbsdf {

constexpr int kEncThreads = 256;
constexpr float kEncSlope = 0.01f;

// out[j] = act(b[j] + sum_k Wt[k][j] in[k] (+ skip[j])), j < n_out; in/out/skip in shared memory
template <bool kAct>
__device__ __forceinline__ void enc_layer(const float* __restrict__ Wt, const float* __restrict__ b, int n_in, int n_out,
                                          const float* in, const float* skip, float* out, float* part)
{
    const int tid = threadIdx.x;
    const int groups = kEncThreads / n_out;              // n_out in {8, ..., 256} divides 256
    const int g = tid / n_out, j = tid - g * n_out;
    const int per = (n_in + groups - 1) / groups;
    const int k0 = g * per, k1 = min(n_in, k0 + per);
    float acc = 0.0f;
    if (g < groups) {
        int k = k0;
        for (; k + 4 <= k1; k += 4) {                    // four independent loads in flight per thread
            const float w0 = __ldg(Wt + (size_t)k * n_out + j), w1 = __ldg(Wt + (size_t)(k + 1) * n_out + j);
            const float w2 = __ldg(Wt + (size_t)(k + 2) * n_out + j), w3 = __ldg(Wt + (size_t)(k + 3) * n_out + j);
            acc = fmaf(w0, in[k], acc);
            acc = fmaf(w1, in[k + 1], acc);
            acc = fmaf(w2, in[k + 2], acc);
            acc = fmaf(w3, in[k + 3], acc);
        }
        for (; k < k1; ++k) acc = fmaf(__ldg(Wt + (size_t)k * n_out + j), in[k], acc);
        part[g * n_out + j] = acc;
    }
    __syncthreads();
    if (tid < n_out) {
        float v = __ldg(b + tid);
        for (int gg = 0; gg < groups; ++gg) v += part[gg * n_out + tid];
        if (skip != nullptr) v += skip[tid];
        out[tid] = kAct ? (v >= 0.0f ? v : kEncSlope * v) : v;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kEncThreads) encode_latent_kernel(const float* __restrict__ w, const float* __restrict__ x_in,
                                                                    int Fr, int He, int L, float* __restrict__ z_row)
{
    extern __shared__ float sm[];
    float* x = sm;                       // Fr + 2
    float* e0 = x + Fr + 2;              // He
    float* r = e0 + He;                  // He
    float* e2 = r + He;                  // He
    float* part = e2 + He;               // 256
    float* z = part + kEncThreads;       // L
    for (int i = threadIdx.x; i < Fr + 2; i += kEncThreads) x[i] = x_in[i];
    __syncthreads();
    const float* E0 = w;
    const float* b0 = E0 + (size_t)(Fr + 2) * He;
    const float* E1 = b0 + He;
    const float* b1 = E1 + (size_t)He * He;
    const float* E2 = b1 + He;
    const float* b2 = E2 + (size_t)He * He;
    const float* E3 = b2 + He;
    const float* b3 = E3 + (size_t)He * L;
    enc_layer<true>(E0, b0, Fr + 2, He, x, nullptr, e0, part);
    enc_layer<true>(E1, b1, He, He, e0, nullptr, r, part);
    enc_layer<true>(E2, b2, He, He, r, e0, e2, part);          // + e0 before the last leaky ReLU
    enc_layer<false>(E3, b3, He, L, e2, nullptr, z, part);
    if (threadIdx.x < L) z_row[threadIdx.x] = z[threadIdx.x];
}

size_t encoder_blob_floats(int Fr, int He, int L)
{
    return (size_t)(Fr + 2) * He + He + 2 * ((size_t)He * He + He) + (size_t)He * L + L;
}

// host weights (row-major [out][in]) -> one blob of transposed matrices [in][out], each followed by its bias
void pack_encoder(int Fr, int He, int L, const nbsdf_encoder_weights* w, float* blob)
{
    const int n_in[4] = { Fr + 2, He, He, He }, n_out[4] = { He, He, He, L };
    size_t off = 0;
    for (int l = 0; l < 4; ++l) {
        for (int k = 0; k < n_in[l]; ++k)
            for (int o = 0; o < n_out[l]; ++o) blob[off + (size_t)k * n_out[l] + o] = w->W[l][(size_t)o * n_in[l] + k];
        off += (size_t)n_in[l] * n_out[l];
        for (int o = 0; o < n_out[l]; ++o) blob[off + o] = w->b[l][o];
        off += n_out[l];
    }
}

cudaError_t launch_encode_latent(const float* w, const float* x_in, int Fr, int He, int L, float* z_row, cudaStream_t s)
{
    const size_t smem = (size_t)(Fr + 2 + 3 * He + kEncThreads + L) * sizeof(float);
    encode_latent_kernel<<<1, kEncThreads, smem, s>>>(w, x_in, Fr, He, L, z_row);
    return cudaGetLastError();
}

}  // namespace nbsdf
