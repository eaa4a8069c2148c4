/* Memory / undefined-behaviour check of the ORACLE ("-fsanitize=address,undefined on the oracle"):
 * built by tests/test_oracle_sanitizers.py together with oracle/*.c under AddressSanitizer + UBSan and run on small
 * inputs that exercise every entry point, frames, background rows, both light types, emitter normals, ranges of a frame,
 * the per-pixel albedo plane and the encoder tail.  Exit code 0 and no sanitizer report = pass. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

typedef struct { int32_t latent_dim, hidden, feat_dim, n_materials; } dims_t;
typedef struct { float u, v, footprint; int32_t material; float wi[3], wo[3]; } query_t;
typedef struct { int32_t type; float vec[3], rgb[3], emit_n[3]; } light_t;
typedef struct { int32_t feat_width, hidden, latent_dim; } enc_dims_t;

int oracle_eval(const dims_t*, const float* const*, const float* const*, const float*, const query_t*, const float*, int64_t, double*, int);
int oracle_shade_frame(const dims_t*, const float* const*, const float* const*, const float*, const float*, const float*,
                       const float*, const int32_t*, int64_t, int64_t, const float*, const light_t*, int, double*, int);
int oracle_pd_eval(const dims_t*, const float* const*, const float* const*, const float*, const float*, const query_t*,
                   const float*, int64_t, double*, double*, int);
int oracle_pd_shade_frame_px(const dims_t*, const float* const*, const float* const*, const float*, const float*, const float*,
                             const float*, const float*, const float*, const int32_t*, int64_t, int64_t, const float*,
                             const light_t*, int, double*, int);
int oracle_encode_latent(const enc_dims_t*, const float* const*, const float* const*, const float*, double, double, double*);

static uint32_t st = 99u;
static float ur(void) { st = st * 1664525u + 1013904223u; return (float)(st >> 8) / 16777216.0f; }
static float* rnd(size_t n, float lo, float hi) { float* p = (float*)malloc(sizeof(float) * n); for (size_t i = 0; i < n; ++i) p[i] = lo + (hi - lo) * ur(); return p; }

int main(void)
{
    enum { L = 8, H = 32, F = 32, M = 3, N = 37, NPX = 45 };
    const int ki[6] = { L + 3, H, H, F + 6, H, H }, ko[6] = { H, H, F, H, H, 3 };
    float *W[6], *b[6];
    for (int l = 0; l < 6; ++l) { W[l] = rnd((size_t)ki[l] * ko[l], -0.3f, 0.3f); b[l] = rnd(ko[l], -0.1f, 0.1f); }
    float* Z = rnd(M * L, -1.0f, 1.0f);
    query_t* q = (query_t*)malloc(sizeof(query_t) * N);
    for (int i = 0; i < N; ++i) {
        q[i].u = 5.0f * ur() - 2.0f; q[i].v = ur(); q[i].footprint = i == 3 ? -1.0f : exp2f(-8.0f * ur()); q[i].material = i == 5 ? -1 : i % M;
        for (int c = 0; c < 3; ++c) { q[i].wi[c] = ur(); q[i].wo[c] = ur(); }
    }
    float* frames = rnd(6 * N, -1.0f, 1.0f);
    for (int c = 0; c < 3; ++c) frames[6 + 3 + c] = 2.0f * frames[6 + c];          /* degenerate tangent hint */
    double* out = (double*)malloc(sizeof(double) * 3 * (N > NPX ? N : NPX));
    dims_t d = { L, H, F, M };
    if (oracle_eval(&d, (const float* const*)W, (const float* const*)b, Z, q, NULL, N, out, 2)) return 1;
    if (oracle_eval(&d, (const float* const*)W, (const float* const*)b, Z, q, frames, N, out, 1)) return 1;
    if (oracle_eval(&d, (const float* const*)W, (const float* const*)b, Z, q, NULL, 0, out, 1)) return 1;
    float *pos = rnd(4 * NPX, -0.5f, 0.5f), *nrm = rnd(4 * NPX, 0.1f, 1.0f), *tan = rnd(4 * NPX, -1.0f, 1.0f);
    int32_t* mat = (int32_t*)malloc(sizeof(int32_t) * NPX);
    for (int p = 0; p < NPX; ++p) { mat[p] = p == 7 ? -1 : p % M; pos[4 * p + 3] = 0.01f + ur(); }
    const float cam[3] = { 0.0f, 0.0f, 1.0f };
    light_t lt[3] = { { 0, { 0.3f, 0.2f, 1.0f }, { 1, 1, 1 }, { 0, 0, 0 } }, { 1, { 0.4f, -0.3f, 0.6f }, { 0.5f, 0.6f, 0.4f }, { 0, 0.6f, -0.8f } },
                      { 1, { 0.1f, 0.2f, -0.7f }, { 0.3f, 0.3f, 0.3f }, { 0, 0, 0 } } };
    if (oracle_shade_frame(&d, (const float* const*)W, (const float* const*)b, Z, pos, nrm, tan, mat, 0, NPX, cam, lt, 3, out, 2)) return 2;
    if (oracle_shade_frame(&d, (const float* const*)W, (const float* const*)b, Z, pos, nrm, tan, mat, 11, 5, cam, lt, 3, out, 1)) return 2;
    if (oracle_shade_frame(&d, (const float* const*)W, (const float* const*)b, Z, pos, nrm, tan, mat, 0, NPX, cam, NULL, 0, out, 1)) return 2;

    /* paper-structured decoder: latent 64, seven layers */
    enum { PL = 64, PH = 16, PF = 8 };
    const int pi[7] = { PL + 24, PH, PF + 5, PH, PH, PH, PH }, po[7] = { PH, PF, PH, PH, PH, PH, 4 };
    float *PW[7], *Pb[7];
    for (int l = 0; l < 7; ++l) { PW[l] = rnd((size_t)pi[l] * po[l], -0.3f, 0.3f); Pb[l] = rnd(po[l], -0.1f, 0.1f); }
    float *PZ = rnd(M * PL, -1.0f, 1.0f), *alb = rnd(M * 12, 0.1f, 0.9f), *apx = rnd(NPX * 12, 0.1f, 0.9f);
    dims_t pd = { PL, PH, PF, M };
    double* comp = (double*)malloc(sizeof(double) * 4 * N);
    for (int i = 0; i < N; ++i) { q[i].footprint = 6.0f * ur() - 0.5f; q[i].wi[2] = ur() - 0.5f; }
    if (oracle_pd_eval(&pd, (const float* const*)PW, (const float* const*)Pb, PZ, alb, q, frames, N, out, comp, 2)) return 3;
    if (oracle_pd_eval(&pd, (const float* const*)PW, (const float* const*)Pb, PZ, alb, q, NULL, N, out, NULL, 1)) return 3;
    if (oracle_pd_shade_frame_px(&pd, (const float* const*)PW, (const float* const*)Pb, PZ, alb, NULL, pos, nrm, tan, mat, 0, NPX, cam, lt, 3, out, 2)) return 4;
    if (oracle_pd_shade_frame_px(&pd, (const float* const*)PW, (const float* const*)Pb, PZ, alb, apx, pos, nrm, tan, mat, 3, 20, cam, lt, 3, out, 1)) return 4;

    /* encoder tail */
    enum { FR = 11, HE = 8, EL = 5 };
    const int ei[4] = { FR + 2, HE, HE, HE }, eo[4] = { HE, HE, HE, EL };
    float *EW[4], *Eb[4];
    for (int l = 0; l < 4; ++l) { EW[l] = rnd((size_t)ei[l] * eo[l], -0.5f, 0.5f); Eb[l] = rnd(eo[l], -0.5f, 0.5f); }
    float* feat = rnd(FR, 0.0f, 1.0f);
    enc_dims_t ed = { FR, HE, EL };
    double z[EL];
    if (oracle_encode_latent(&ed, (const float* const*)EW, (const float* const*)Eb, feat, 0.3, 1.2, z)) return 5;
    enc_dims_t e0 = { 0, HE, EL };      /* no feature at all: x = [alpha, beta] */
    float* EW0 = rnd((size_t)2 * HE, -0.5f, 0.5f);
    const float* EWz[4] = { EW0, EW[1], EW[2], EW[3] };
    if (oracle_encode_latent(&e0, EWz, (const float* const*)Eb, NULL, 0.3, 1.2, z)) return 5;
    double s = 0.0;
    for (int i = 0; i < EL; ++i) s += z[i];
    printf("OK %g\n", s + out[0]);
    return 0;
}
