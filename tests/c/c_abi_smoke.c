/* A C caller of the C ABI (include/nbsdf.h): no Python, no torch -- CUDA runtime for device memory, libnbsdf.so for the
 * hot path, liboracle.so (test infrastructure) for the expected values.  Built and run by tests/test_gpu_c_abi.py.
 * Network: BASELINE.json configs[0] shapes (L16, H64, F32), weights from a small LCG; 1000 queries + a 40x25 frame.
 * Prints "OK max_rel_eval=... max_rel_frame=..." and exits 0 when both are within the fp16 tolerance (1e-2). */
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "nbsdf.h"

/* oracle/nbsdf_oracle.c */
typedef struct { int32_t latent_dim, hidden, feat_dim, n_materials; } oracle_dims;
int oracle_eval(const oracle_dims* d, const float* const* W, const float* const* b, const float* Z, const nbsdf_query* q,
                const float* frames, int64_t n, double* out, int n_threads);
int oracle_shade_frame(const oracle_dims* d, const float* const* W, const float* const* b, const float* Z, const float* pos_fp,
                       const float* nrm_u, const float* tan_v, const int32_t* material, int64_t first, int64_t count,
                       const float* cam_pos, const nbsdf_light* lights, int n_lights, double* out, int n_threads);

static uint32_t lcg_state = 12345u;
static float urand(void) { lcg_state = lcg_state * 1664525u + 1013904223u; return (float)(lcg_state >> 8) / 16777216.0f; }

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA %s: %s\n", #x, cudaGetErrorString(e_)); return 2; } } while (0)
#define NB(x) do { int rc_ = (x); if (rc_ != NBSDF_OK) { printf("nbsdf %s: %d %s\n", #x, rc_, nbsdf_last_error(ctx)); return 3; } } while (0)

int main(void)
{
    enum { L = 16, H = 64, F = 32, M = 4, N = 1000, WPX = 40, HPX = 25, NPX = WPX * HPX };
    const int n_in[6] = { L + 3, H, H, F + 6, H, H }, n_out[6] = { H, H, F, H, H, 3 };
    float* W[6]; float* b[6];
    for (int l = 0; l < 6; ++l) {
        const float a = sqrtf(6.0f / (float)(n_in[l] + n_out[l]));
        W[l] = (float*)malloc(sizeof(float) * n_in[l] * n_out[l]);
        b[l] = (float*)malloc(sizeof(float) * n_out[l]);
        for (int i = 0; i < n_in[l] * n_out[l]; ++i) {
            /* bf16-representable weights ("stored in bf16"): drop the low 16 bits */
            union { float f; uint32_t u; } v; v.f = (2.0f * urand() - 1.0f) * a; v.u &= 0xffff0000u; W[l][i] = v.f;
        }
        for (int i = 0; i < n_out[l]; ++i) b[l][i] = 0.02f * (urand() - 0.5f);
    }
    float Z[M * L];
    for (int i = 0; i < M * L; ++i) Z[i] = 2.0f * urand() - 1.0f;
    nbsdf_query* q = (nbsdf_query*)malloc(sizeof(nbsdf_query) * N);
    for (int i = 0; i < N; ++i) {
        q[i].u = 3.0f * urand() - 1.0f; q[i].v = urand(); q[i].footprint = exp2f(-8.0f * urand()); q[i].material = (int32_t)(urand() * M) % M;
        float r = sqrtf(urand()), ph = 6.2831853f * urand();
        q[i].wi[0] = r * cosf(ph); q[i].wi[1] = r * sinf(ph); q[i].wi[2] = sqrtf(1.0f - r * r);
        r = sqrtf(urand()); ph = 6.2831853f * urand();
        q[i].wo[0] = r * cosf(ph); q[i].wo[1] = r * sinf(ph); q[i].wo[2] = sqrtf(1.0f - r * r);
    }
    if (N > 7) q[7].material = -1;

    nbsdf_config cfg = { L, H, F, M, NBSDF_PREC_FP16, 0 };
    nbsdf_weights w;
    for (int l = 0; l < 6; ++l) { w.W[l] = W[l]; w.b[l] = b[l]; }
    nbsdf_ctx* ctx = NULL;
    NB(nbsdf_create(&cfg, &w, &ctx));
    cudaStream_t s;
    CK(cudaStreamCreate(&s));
    NB(nbsdf_set_latents(ctx, 0, M, Z, s));

    /* ---- nbsdf_eval ---- */
    nbsdf_query* q_dev; float* rgb_dev;
    CK(cudaMalloc((void**)&q_dev, sizeof(nbsdf_query) * N));
    CK(cudaMalloc((void**)&rgb_dev, sizeof(float) * 3 * N));
    CK(cudaMemcpyAsync(q_dev, q, sizeof(nbsdf_query) * N, cudaMemcpyHostToDevice, s));
    NB(nbsdf_eval(ctx, q_dev, NULL, N, rgb_dev, s));
    float* rgb = (float*)malloc(sizeof(float) * 3 * N);
    CK(cudaMemcpyAsync(rgb, rgb_dev, sizeof(float) * 3 * N, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    oracle_dims od = { L, H, F, M };
    double* ref = (double*)malloc(sizeof(double) * 3 * N);
    if (oracle_eval(&od, (const float* const*)W, (const float* const*)b, Z, q, NULL, N, ref, 1) != 0) { printf("oracle_eval failed\n"); return 4; }
    double max_eval = 0.0;
    for (int i = 0; i < 3 * N; ++i) {
        const double d = fabs((double)rgb[i] - ref[i]) / fmax(fabs(ref[i]), 1e-6);
        if (!(d <= max_eval)) max_eval = d;
    }
    if (rgb[21] != 0.0f || rgb[22] != 0.0f || rgb[23] != 0.0f) { printf("background query is not black\n"); return 5; }

    /* ---- nbsdf_shade_frame ---- */
    float* pos = (float*)malloc(sizeof(float) * 4 * NPX); float* nrm = (float*)malloc(sizeof(float) * 4 * NPX);
    float* tan = (float*)malloc(sizeof(float) * 4 * NPX); int32_t* mat = (int32_t*)malloc(sizeof(int32_t) * NPX);
    for (int p = 0; p < NPX; ++p) {
        pos[4 * p] = (float)(p % WPX) / WPX - 0.5f; pos[4 * p + 1] = (float)(p / WPX) / HPX - 0.5f; pos[4 * p + 2] = 0.0f; pos[4 * p + 3] = 0.01f;
        const float a = 0.5f * urand(), ph = 6.2831853f * urand();
        nrm[4 * p] = sinf(a) * cosf(ph); nrm[4 * p + 1] = sinf(a) * sinf(ph); nrm[4 * p + 2] = cosf(a); nrm[4 * p + 3] = 12.0f * urand();
        tan[4 * p] = 1.0f; tan[4 * p + 1] = 0.0f; tan[4 * p + 2] = 0.0f; tan[4 * p + 3] = 12.0f * urand();
        mat[p] = p % M;
    }
    nbsdf_light lights[2] = { { 0, { 0.3f, 0.2f, 1.0f }, { 1.0f, 1.0f, 1.0f }, { 0.0f, 0.0f, 0.0f } },
                              { 1, { 0.4f, -0.3f, 0.6f }, { 0.5f, 0.6f, 0.4f }, { 0.0f, 0.6f, -0.8f } } };
    float *pos_d, *nrm_d, *tan_d, *rad_d; int32_t* mat_d;
    CK(cudaMalloc((void**)&pos_d, sizeof(float) * 4 * NPX)); CK(cudaMalloc((void**)&nrm_d, sizeof(float) * 4 * NPX));
    CK(cudaMalloc((void**)&tan_d, sizeof(float) * 4 * NPX)); CK(cudaMalloc((void**)&mat_d, sizeof(int32_t) * NPX));
    CK(cudaMalloc((void**)&rad_d, sizeof(float) * 3 * NPX));
    CK(cudaMemcpy(pos_d, pos, sizeof(float) * 4 * NPX, cudaMemcpyHostToDevice)); CK(cudaMemcpy(nrm_d, nrm, sizeof(float) * 4 * NPX, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(tan_d, tan, sizeof(float) * 4 * NPX, cudaMemcpyHostToDevice)); CK(cudaMemcpy(mat_d, mat, sizeof(int32_t) * NPX, cudaMemcpyHostToDevice));
    nbsdf_gbuffer g = { pos_d, nrm_d, tan_d, mat_d, WPX, HPX, { 0.0f, 0.0f, 1.0f }, NULL };
    NB(nbsdf_shade_frame(ctx, &g, lights, 2, rad_d, s));
    float* rad = (float*)malloc(sizeof(float) * 3 * NPX);
    CK(cudaMemcpyAsync(rad, rad_d, sizeof(float) * 3 * NPX, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    double* fref = (double*)malloc(sizeof(double) * 3 * NPX);
    const float cam[3] = { 0.0f, 0.0f, 1.0f };
    if (oracle_shade_frame(&od, (const float* const*)W, (const float* const*)b, Z, pos, nrm, tan, mat, 0, NPX, cam, lights, 2, fref, 1) != 0) { printf("oracle_shade_frame failed\n"); return 4; }
    double max_frame = 0.0;
    for (int i = 0; i < 3 * NPX; ++i) {
        const double d = fabs((double)rad[i] - fref[i]) / fmax(fabs(fref[i]), 1e-6);
        if (!(d <= max_frame)) max_frame = d;
    }
    if (nbsdf_launch_count(ctx) != 2) { printf("launch count %lld\n", (long long)nbsdf_launch_count(ctx)); return 6; }
    if (nbsdf_eval(ctx, NULL, NULL, 5, rgb_dev, s) != NBSDF_E_INVALID) { printf("NULL queries were accepted\n"); return 7; }
    nbsdf_destroy(ctx);
    if (!(max_eval <= 1e-2) || !(max_frame <= 1e-2)) { printf("FAIL max_rel_eval=%.3e max_rel_frame=%.3e\n", max_eval, max_frame); return 1; }
    printf("OK max_rel_eval=%.3e max_rel_frame=%.3e\n", max_eval, max_frame);
    return 0;
}
