/*
 * nbsdf_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU definition of the neural woven-fabric BSDF decoder hot path
 * (arXiv 2406.17782, "Real-time Neural Woven Fabric Rendering").  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code, header, table or helper with the CUDA
 * library (paper_2406_17782_b200/csrc); the record layouts below restate the
 * wire format of the inputs, nothing else.
 *
 * What it computes (each step cites the passage it follows):
 *   - decoder data flow: the material latent z is fused with the spatial query
 *     (footprint position + size) by a small MLP into a spatial feature, which is
 *     concatenated with the angular inputs (wi, wo) and decoded by a second MLP
 *     -- PAPER.md:164 (sec. 4.2 "Decoder"), signature PAPER.md:160, Eq. 7 at 149.
 *   - shapes/activations: BASELINE.json configs[0..3] (latent L, raw [u,v,log2 fp],
 *     2 ReLU hidden layers of H to an F-d linear feature; [feat, wi3, wo3] through
 *     2 ReLU hidden layers of H to 3 softplus outputs).  DESIGN.md "Readings" lists
 *     every place this differs from the paper's own hyper-parameters.
 *   - per-frame recipe: "prepare the query (wi, wo, P) and compute the lighting ...
 *     infer the decoder ... multiply it by the lighting" -- PAPER.md:196 (sec. 4.3);
 *     point or directional lights, direct illumination only -- PAPER.md:232.
 *
 * The oracle is the plain definition: every W x is the naive double loop in index
 * order, in double, on fp32 inputs promoted exactly.  No blocking, no fusion, no
 * reuse of MLP-A across lights (the reuse in the CUDA path is itself under test).
 * OpenMP only splits the independent queries/pixels across threads.
 *
 * Pins: tests/test_oracle_pins.py (hand-computed 1-hidden-unit networks, softplus
 * closed-form values, zero-weight layers, ReLU-transparent affine case against an
 * independent naive matmul, uv periodicity, log-footprint exact powers of two,
 * frame worked example + rotation invariance, latent indirection, shading closed
 * forms and linearity).  Agreement with the paper's *trained* network is
 * "parity unpinned": the paper prints no numeric decoder input/output pair and its
 * weights are not available.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t latent_dim;   /* L */
    int32_t hidden;       /* H */
    int32_t feat_dim;     /* F */
    int32_t n_materials;  /* M */
} oracle_dims;

/* 40-byte query record: u, v, footprint, material, wi[3], wo[3] */
typedef struct {
    float u, v, footprint;
    int32_t material;
    float wi[3];
    float wo[3];
} oracle_query;

/* 40-byte light record: type 0 = directional (vec = direction TO the light),
 * type 1 = point (vec = position); rgb = radiance (dir.) or intensity (point);
 * emit_n = emitter normal of a point light, (0,0,0) = isotropic. */
typedef struct {
    int32_t type;
    float vec[3];
    float rgb[3];
    float emit_n[3];
} oracle_light;

/* B7: softplus(x) = ln(1 + e^x), beta = 1, no threshold; stable two-branch form. */
double oracle_softplus(double x)
{
    return x > 0.0 ? x + log1p(exp(-x)) : log1p(exp(x));
}

/* A2: wrap to the pattern period (period 1 in uv units). */
double oracle_wrap(double u)
{
    return u - floor(u);
}

/* A3: log2 of the footprint side length, clamped to [2^-20, 2^4]. */
double oracle_log_footprint(double fp)
{
    const double lo = ldexp(1.0, -20), hi = 16.0;
    double c = fp;
    if (!(c > lo)) c = lo;      /* also catches fp <= 0 */
    if (c > hi) c = hi;
    return log2(c);
}

/* A4: orthonormal frame from (n, t): n^ = n/|n|; t' = t - n^(n^.t); degenerate t' is
 * replaced by e_k - n^ n^_k with k = argmin |n^_k| (lowest k on ties); b^ = n^ x t^.
 * Writes w_loc = (w.t^, w.b^, w.n^). */
void oracle_to_local(const double n_in[3], const double t_in[3], const double w[3], double w_loc[3])
{
    double n[3], t[3], b[3];
    double nn = sqrt(n_in[0] * n_in[0] + n_in[1] * n_in[1] + n_in[2] * n_in[2]);
    for (int i = 0; i < 3; ++i) n[i] = n_in[i] / nn;
    double nt = n[0] * t_in[0] + n[1] * t_in[1] + n[2] * t_in[2];
    for (int i = 0; i < 3; ++i) t[i] = t_in[i] - n[i] * nt;
    double tt = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
    if (tt < 1e-12) {
        int k = 0;
        for (int i = 1; i < 3; ++i)
            if (fabs(n[i]) < fabs(n[k])) k = i;
        for (int i = 0; i < 3; ++i) t[i] = (i == k ? 1.0 : 0.0) - n[i] * n[k];
        tt = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
    }
    double tl = sqrt(tt);
    for (int i = 0; i < 3; ++i) t[i] /= tl;
    b[0] = n[1] * t[2] - n[2] * t[1];
    b[1] = n[2] * t[0] - n[0] * t[2];
    b[2] = n[0] * t[1] - n[1] * t[0];
    w_loc[0] = w[0] * t[0] + w[1] * t[1] + w[2] * t[2];
    w_loc[1] = w[0] * b[0] + w[1] * b[1] + w[2] * b[2];
    w_loc[2] = w[0] * n[0] + w[1] * n[1] + w[2] * n[2];
}

/* y = W x + b, W row-major [n_out][n_in], naive loops in index order. */
static void affine(const float* W, const float* b, int n_out, int n_in, const double* x, double* y)
{
    for (int o = 0; o < n_out; ++o) {
        double acc = 0.0;
        for (int i = 0; i < n_in; ++i) acc += (double)W[(size_t)o * n_in + i] * x[i];
        y[o] = acc + (double)b[o];
    }
}

static void relu_inplace(double* x, int n)
{
    for (int i = 0; i < n; ++i) x[i] = x[i] > 0.0 ? x[i] : 0.0;
}

/* One decoder evaluation (steps 1-7 of DESIGN.md "Oracle").  wi, wo already local.
 * scratch holds at least (L+3) + 2H + (F+6) + 3 doubles. */
static void decoder(const oracle_dims* d, const float* const W[6], const float* const b[6],
                    const float* Z, int material, double u, double v, double footprint,
                    const double wi[3], const double wo[3], double* scratch, double rgb[3])
{
    const int L = d->latent_dim, H = d->hidden, F = d->feat_dim;
    double* x = scratch;            /* L+3 */
    double* h1 = x + (L + 3);       /* H */
    double* h2 = h1 + H;            /* H */
    double* y = h2 + H;             /* F+6 */
    double* o = y + (F + 6);        /* 3 */

    /* spatial input x = [z, u', v', lf]  (latent fused with position and size of P) */
    for (int i = 0; i < L; ++i) x[i] = (double)Z[(size_t)material * L + i];
    x[L + 0] = oracle_wrap(u);
    x[L + 1] = oracle_wrap(v);
    x[L + 2] = oracle_log_footprint(footprint);

    /* MLP-A: two ReLU hidden layers, linear feature */
    affine(W[0], b[0], H, L + 3, x, h1);  relu_inplace(h1, H);
    affine(W[1], b[1], H, H, h1, h2);     relu_inplace(h2, H);
    affine(W[2], b[2], F, H, h2, y);      /* feat -> y[0..F) */

    /* angular input y = [feat, wi, wo]  ("concatenate it with the angular parameters") */
    for (int i = 0; i < 3; ++i) { y[F + i] = wi[i]; y[F + 3 + i] = wo[i]; }

    /* MLP-B: two ReLU hidden layers, 3 outputs, softplus */
    affine(W[3], b[3], H, F + 6, y, h1);  relu_inplace(h1, H);
    affine(W[4], b[4], H, H, h1, h2);     relu_inplace(h2, H);
    affine(W[5], b[5], 3, H, h2, o);
    for (int c = 0; c < 3; ++c) rgb[c] = oracle_softplus(o[c]);
}

static size_t scratch_len(const oracle_dims* d)
{
    return (size_t)(d->latent_dim + 3) + 2 * (size_t)d->hidden + (size_t)(d->feat_dim + 6) + 3;
}

/* Batched evaluation.  frames: [n][6] = (n, t) per query, or NULL when wi/wo are
 * already local.  out: [n][3] doubles.  Returns 0, or -1 on bad arguments. */
int oracle_eval(const oracle_dims* d, const float* const W[6], const float* const b[6], const float* Z,
                const oracle_query* q, const float* frames, int64_t n, double* out, int n_threads)
{
    if (!d || !W || !b || !Z || n < 0 || (n > 0 && (!q || !out))) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    const size_t sl = scratch_len(d);
#pragma omp parallel
    {
        double* scratch = (double*)malloc(sl * sizeof(double));
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double* rgb = out + 3 * i;
            if (q[i].material < 0) { rgb[0] = rgb[1] = rgb[2] = 0.0; continue; }
            double wi[3] = { q[i].wi[0], q[i].wi[1], q[i].wi[2] };
            double wo[3] = { q[i].wo[0], q[i].wo[1], q[i].wo[2] };
            if (frames) {
                const float* f = frames + 6 * i;
                double nn[3] = { f[0], f[1], f[2] }, tt[3] = { f[3], f[4], f[5] }, a[3], c[3];
                oracle_to_local(nn, tt, wi, a);
                oracle_to_local(nn, tt, wo, c);
                memcpy(wi, a, sizeof a); memcpy(wo, c, sizeof c);
            }
            decoder(d, W, b, Z, q[i].material, q[i].u, q[i].v, q[i].footprint, wi, wo, scratch, rgb);
        }
        free(scratch);
    }
    return 0;
}

/* Frame shading (C1-C3).  G-buffer planes are HOST arrays here:
 *   pos_fp [h*w][4] = x, y, z, footprint;  nrm_u [h*w][4] = nx, ny, nz, u;
 *   tan_v [h*w][4] = tx, ty, tz, v;  material [h*w] (< 0 = background -> 0).
 * Per pixel: wo = normalize(cam - x); for each light in index order
 *   directional: wi = vec/|vec|, E = rgb
 *   point:       v = vec - x, wi = v/|v|, E = rgb * max(0, -wi.emit_n) / |v|^2   (emit_n = 0 -> factor 1)
 *   L += decoder(..., wi_loc, wo_loc) * E * max(0, wi_loc.z)
 * The full decoder is evaluated per (pixel, light).  Pixels [first, first+count). */
int oracle_shade_frame(const oracle_dims* d, const float* const W[6], const float* const b[6], const float* Z,
                       const float* pos_fp, const float* nrm_u, const float* tan_v, const int32_t* material,
                       int64_t first, int64_t count, const float cam_pos[3],
                       const oracle_light* lights, int n_lights, double* out, int n_threads)
{
    if (!d || !W || !b || !Z || count < 0 || n_lights < 0) return -1;
    if (count > 0 && (!pos_fp || !nrm_u || !tan_v || !material || !out || !cam_pos)) return -1;
    if (n_lights > 0 && !lights) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    const size_t sl = scratch_len(d);
#pragma omp parallel
    {
        double* scratch = (double*)malloc(sl * sizeof(double));
#pragma omp for schedule(static)
        for (int64_t k = 0; k < count; ++k) {
            const int64_t p = first + k;
            double* Lp = out + 3 * k;
            Lp[0] = Lp[1] = Lp[2] = 0.0;
            const int m = material[p];
            if (m < 0) continue;
            const double x[3] = { pos_fp[4 * p], pos_fp[4 * p + 1], pos_fp[4 * p + 2] };
            const double fp = pos_fp[4 * p + 3];
            const double nn[3] = { nrm_u[4 * p], nrm_u[4 * p + 1], nrm_u[4 * p + 2] };
            const double u = nrm_u[4 * p + 3];
            const double tt[3] = { tan_v[4 * p], tan_v[4 * p + 1], tan_v[4 * p + 2] };
            const double v = tan_v[4 * p + 3];
            double wo[3] = { cam_pos[0] - x[0], cam_pos[1] - x[1], cam_pos[2] - x[2] };
            double wl = sqrt(wo[0] * wo[0] + wo[1] * wo[1] + wo[2] * wo[2]);
            for (int i = 0; i < 3; ++i) wo[i] /= wl;
            double wo_loc[3];
            oracle_to_local(nn, tt, wo, wo_loc);
            for (int l = 0; l < n_lights; ++l) {
                double wi[3], E[3];
                if (lights[l].type == 0) {
                    double dl = sqrt((double)lights[l].vec[0] * lights[l].vec[0] +
                                     (double)lights[l].vec[1] * lights[l].vec[1] +
                                     (double)lights[l].vec[2] * lights[l].vec[2]);
                    for (int i = 0; i < 3; ++i) { wi[i] = lights[l].vec[i] / dl; E[i] = lights[l].rgb[i]; }
                } else {
                    double vv[3] = { lights[l].vec[0] - x[0], lights[l].vec[1] - x[1], lights[l].vec[2] - x[2] };
                    double d2 = vv[0] * vv[0] + vv[1] * vv[1] + vv[2] * vv[2];
                    double dl = sqrt(d2);
                    for (int i = 0; i < 3; ++i) wi[i] = vv[i] / dl;
                    double en[3] = { lights[l].emit_n[0], lights[l].emit_n[1], lights[l].emit_n[2] };
                    double fac = 1.0;
                    if (en[0] != 0.0 || en[1] != 0.0 || en[2] != 0.0) {
                        double c = -(wi[0] * en[0] + wi[1] * en[1] + wi[2] * en[2]);
                        fac = c > 0.0 ? c : 0.0;
                    }
                    for (int i = 0; i < 3; ++i) E[i] = lights[l].rgb[i] * fac / d2;
                }
                double wi_loc[3], rgb[3];
                oracle_to_local(nn, tt, wi, wi_loc);
                double c = wi_loc[2] > 0.0 ? wi_loc[2] : 0.0;
                decoder(d, W, b, Z, m, u, v, fp, wi_loc, wo_loc, scratch, rgb);
                for (int i = 0; i < 3; ++i) Lp[i] += rgb[i] * E[i] * c;
            }
        }
        free(scratch);
    }
    return 0;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
