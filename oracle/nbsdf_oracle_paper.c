/*
 * nbsdf_oracle_paper.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU definition of the decoder with the PAPER'S OWN structure, next to
 * the BASELINE.json-shaped decoder of nbsdf_oracle.c.  Same rules: only tests/, smoke() and bench.py's CPU legs may
 * call it; it shares nothing with the CUDA library.
 *
 * What it computes, step by step in the paper's order (PAPER.md line / section / equation):
 *   1. material latent z of size 64                                           PAPER.md:162 (sec. 4.2 "Encoder")
 *   2. one-blob encoding of the footprint position (2) and size (1), 3 -> 24   PAPER.md:164, 244 (sec. 4.2, 6.2)
 *      channels = 8 bins per scalar.  The paper cites Mueller et al. and gives no formula; reading:
 *      a Gaussian of sigma = 1/k centred at the scalar s in [0,1], sampled at the k bin centres (i + 1/2)/k.
 *      Position is wrapped to the pattern period; size (multiples of the pattern size L_t, range
 *      (0,5), Table 2) is clamped to [0,5] and divided by 5.
 *   3. fusion: "two fully connected layers to fuse the material latent vector with the spatial parameters to get
 *      a spatial feature"
 *   4. angular decoder: [feature, wi (x,y,z), wo (x,y)] through "five fully connected layers with one skip
 *      connection"; the residual block is "two fully connected layers and a skip connection before the last leaky
 *      ReLU"                                                                   PAPER.md:164, 168 (Fig. 3 caption)
 *      Reading: D1, then the block [D2, lrelu, D3, + D1's output, lrelu], then D4, D5; leaky ReLU (slope 0.01,
 *      unstated in the paper) after every layer but the last.
 *   5. four outputs (C_warp, C_weft, S_warp, S_weft)                           PAPER.md:149 (Eq. 7)
 *      the specular pair is predicted through g(x) = ln(k x + 1), k = 100 for BRDF and 1000 for BTDF
 *      (Eq. 9), so inference inverts it: S = (e^y - 1) / k, BTDF <=> wi_local.z < 0
 *      ("z ... might be negative for transmission").
 *   6. f = kd_warp C_warp + kd_weft C_weft + ks_warp S_warp + ks_weft S_weft   PAPER.md:154 (Eq. 8), per RGB channel
 *   7. frame: BSDF value x lighting; |cos| instead of max(0, cos) so that transmission contributes.
 * Layer widths are not in the paper: latent 64 is; H (hidden) and F (feature) are parameters here.
 *
 * Pins: tests/test_oracle_paper_pins.py.  Agreement with the paper's trained network: "parity unpinned" (no weights,
 * no printed input/output pair; widths, slope, one-blob kernel and skip position are readings).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* from nbsdf_oracle.c (same library) */
double oracle_wrap(double u);
void oracle_to_local(const double n_in[3], const double t_in[3], const double w[3], double w_loc[3]);

typedef struct {
    int32_t latent_dim;   /* 64 in the paper */
    int32_t hidden;       /* H */
    int32_t feat_dim;     /* F */
    int32_t n_materials;  /* M */
} oracle_pd_dims;

typedef struct {
    float u, v, footprint;     /* footprint = size of P in multiples of the pattern size */
    int32_t material;
    float wi[3];
    float wo[3];               /* only x, y enter the network */
} oracle_pd_query;

typedef struct {
    int32_t type;
    float vec[3];
    float rgb[3];
    float emit_n[3];
} oracle_pd_light;

#define PD_BINS 8
#define PD_SLOPE 0.01

/* step 2: out[i] = exp(-(c_i - s)^2 / (2 sigma^2)), c_i = (i + 1/2)/k, sigma = 1/k */
void oracle_oneblob(double s, int k, double* out)
{
    const double sigma = 1.0 / (double)k;
    for (int i = 0; i < k; ++i) {
        const double c = ((double)i + 0.5) / (double)k;
        const double d = c - s;
        out[i] = exp(-(d * d) / (2.0 * sigma * sigma));
    }
}

double oracle_leaky(double x)
{
    return x > 0.0 ? x : PD_SLOPE * x;
}

/* footprint size -> [0,1] */
double oracle_size01(double size)
{
    double c = size;
    if (!(c > 0.0)) c = 0.0;
    if (c > 5.0) c = 5.0;
    return c / 5.0;
}

/* step 5: inverse of g(x) = ln(k x + 1) */
double oracle_inv_logmap(double y, double k)
{
    return expm1(y) / k;
}

static void pd_affine(const float* W, const float* b, int n_out, int n_in, const double* x, double* y)
{
    for (int o = 0; o < n_out; ++o) {
        double acc = 0.0;
        for (int i = 0; i < n_in; ++i) acc += (double)W[(size_t)o * n_in + i] * x[i];
        y[o] = acc + (double)b[o];
    }
}

static void pd_leaky_inplace(double* x, int n)
{
    for (int i = 0; i < n; ++i) x[i] = oracle_leaky(x[i]);
}

static size_t pd_scratch_len(const oracle_pd_dims* d)
{
    return (size_t)(d->latent_dim + 3 * PD_BINS) + 4 * (size_t)d->hidden + (size_t)(d->feat_dim + 5) + 4;
}

/* One decoder evaluation: the four components (steps 1-5).  wi, wo local.  W/b: 7 layers
 *   0: (L+24) -> H   1: H -> F   2: (F+5) -> H   3: H -> H   4: H -> H (+skip)   5: H -> H   6: H -> 4 */
static void pd_components(const oracle_pd_dims* d, const float* const W[7], const float* const b[7], const float* Z,
                          int material, double u, double v, double size, const double wi[3], const double wo[3],
                          double* scratch, double comp[4])
{
    const int L = d->latent_dim, H = d->hidden, F = d->feat_dim;
    double* x = scratch;                  /* L + 24 */
    double* a1 = x + (L + 3 * PD_BINS);   /* H */
    double* y = a1 + H;                   /* F + 5 */
    double* d1 = y + (F + 5);             /* H */
    double* r = d1 + H;                   /* H */
    double* d3 = r + H;                   /* H */
    double* o = d3 + H;                   /* 4 */

    for (int i = 0; i < L; ++i) x[i] = (double)Z[(size_t)material * L + i];
    oracle_oneblob(oracle_wrap(u), PD_BINS, x + L);
    oracle_oneblob(oracle_wrap(v), PD_BINS, x + L + PD_BINS);
    oracle_oneblob(oracle_size01(size), PD_BINS, x + L + 2 * PD_BINS);

    /* fusion: two FC layers -> spatial feature */
    pd_affine(W[0], b[0], H, L + 3 * PD_BINS, x, a1);  pd_leaky_inplace(a1, H);
    pd_affine(W[1], b[1], F, H, a1, y);                pd_leaky_inplace(y, F);

    /* angular input: feature, wi (3 channels), wo (2 channels) */
    y[F + 0] = wi[0]; y[F + 1] = wi[1]; y[F + 2] = wi[2];
    y[F + 3] = wo[0]; y[F + 4] = wo[1];

    /* angular decoder: D1, residual block (D2, D3, skip from D1's output, before the last leaky ReLU), D4, D5 */
    pd_affine(W[2], b[2], H, F + 5, y, d1);  pd_leaky_inplace(d1, H);
    pd_affine(W[3], b[3], H, H, d1, r);      pd_leaky_inplace(r, H);
    pd_affine(W[4], b[4], H, H, r, d3);
    for (int i = 0; i < H; ++i) d3[i] = oracle_leaky(d3[i] + d1[i]);
    pd_affine(W[5], b[5], H, H, d3, r);      pd_leaky_inplace(r, H);
    pd_affine(W[6], b[6], 4, H, r, o);

    const double k = wi[2] < 0.0 ? 1000.0 : 100.0;
    comp[0] = o[0];
    comp[1] = o[1];
    comp[2] = oracle_inv_logmap(o[2], k);
    comp[3] = oracle_inv_logmap(o[3], k);
}

/* step 6 (Eq. 8).  albedo: [kd_warp rgb, kd_weft rgb, ks_warp rgb, ks_weft rgb] of the material */
static void pd_combine(const float* albedo, const double comp[4], double rgb[3])
{
    for (int c = 0; c < 3; ++c)
        rgb[c] = (double)albedo[c] * comp[0] + (double)albedo[3 + c] * comp[1] +
                 (double)albedo[6 + c] * comp[2] + (double)albedo[9 + c] * comp[3];
}

/* Batched evaluation.  albedos: [M][12].  out_rgb: [n][3]; out_comp: [n][4] or NULL.  frames as in oracle_eval. */
int oracle_pd_eval(const oracle_pd_dims* d, const float* const W[7], const float* const b[7], const float* Z,
                   const float* albedos, const oracle_pd_query* q, const float* frames, int64_t n,
                   double* out_rgb, double* out_comp, int n_threads)
{
    if (!d || !W || !b || !Z || !albedos || n < 0 || (n > 0 && (!q || !out_rgb))) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    const size_t sl = pd_scratch_len(d);
#pragma omp parallel
    {
        double* scratch = (double*)malloc(sl * sizeof(double));
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            double* rgb = out_rgb + 3 * i;
            double comp[4] = { 0.0, 0.0, 0.0, 0.0 };
            if (q[i].material < 0) {
                rgb[0] = rgb[1] = rgb[2] = 0.0;
            } else {
                double wi[3] = { q[i].wi[0], q[i].wi[1], q[i].wi[2] };
                double wo[3] = { q[i].wo[0], q[i].wo[1], q[i].wo[2] };
                if (frames) {
                    const float* f = frames + 6 * i;
                    double nn[3] = { f[0], f[1], f[2] }, tt[3] = { f[3], f[4], f[5] }, a[3], c[3];
                    oracle_to_local(nn, tt, wi, a);
                    oracle_to_local(nn, tt, wo, c);
                    memcpy(wi, a, sizeof a); memcpy(wo, c, sizeof c);
                }
                pd_components(d, W, b, Z, q[i].material, q[i].u, q[i].v, q[i].footprint, wi, wo, scratch, comp);
                pd_combine(albedos + 12 * (size_t)q[i].material, comp, rgb);
            }
            if (out_comp) memcpy(out_comp + 4 * i, comp, sizeof comp);
        }
        free(scratch);
    }
    return 0;
}

/* Frame shading with the paper-structured decoder: as oracle_shade_frame, but L += f * E * |wi_local.z|.
 * albedo_px: NULL, or a per-pixel albedo plane [h*w][12] (kd_warp, kd_weft, ks_warp, ks_weft, RGB each) that replaces the
 * material's table row in Eq. 8 for that pixel -- "spatial-varying appearances when applying albedo maps, by computing
 * k_d and k_s via mipmapping": the mip-mapped fetch is the renderer's, its result is this plane. */
int oracle_pd_shade_frame_px(const oracle_pd_dims* d, const float* const W[7], const float* const b[7], const float* Z,
                             const float* albedos, const float* albedo_px, const float* pos_fp, const float* nrm_u,
                             const float* tan_v, const int32_t* material, int64_t first, int64_t count,
                             const float cam_pos[3], const oracle_pd_light* lights, int n_lights, double* out, int n_threads)
{
    if (!d || !W || !b || !Z || !albedos || count < 0 || n_lights < 0) return -1;
    if (count > 0 && (!pos_fp || !nrm_u || !tan_v || !material || !out || !cam_pos)) return -1;
    if (n_lights > 0 && !lights) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    const size_t sl = pd_scratch_len(d);
#pragma omp parallel
    {
        double* scratch = (double*)malloc(sl * sizeof(double));
#pragma omp for schedule(static)
        for (int64_t kk = 0; kk < count; ++kk) {
            const int64_t p = first + kk;
            double* Lp = out + 3 * kk;
            Lp[0] = Lp[1] = Lp[2] = 0.0;
            const int m = material[p];
            if (m < 0) continue;
            const double x[3] = { pos_fp[4 * p], pos_fp[4 * p + 1], pos_fp[4 * p + 2] };
            const double size = pos_fp[4 * p + 3];
            const double nn[3] = { nrm_u[4 * p], nrm_u[4 * p + 1], nrm_u[4 * p + 2] };
            const double u = nrm_u[4 * p + 3];
            const double tt[3] = { tan_v[4 * p], tan_v[4 * p + 1], tan_v[4 * p + 2] };
            const double v = tan_v[4 * p + 3];
            double wo[3] = { cam_pos[0] - x[0], cam_pos[1] - x[1], cam_pos[2] - x[2] };
            const double wl = sqrt(wo[0] * wo[0] + wo[1] * wo[1] + wo[2] * wo[2]);
            for (int i = 0; i < 3; ++i) wo[i] /= wl;
            double wo_loc[3];
            oracle_to_local(nn, tt, wo, wo_loc);
            for (int l = 0; l < n_lights; ++l) {
                double wi[3], E[3];
                if (lights[l].type == 0) {
                    const double dl = sqrt((double)lights[l].vec[0] * lights[l].vec[0] +
                                           (double)lights[l].vec[1] * lights[l].vec[1] +
                                           (double)lights[l].vec[2] * lights[l].vec[2]);
                    for (int i = 0; i < 3; ++i) { wi[i] = lights[l].vec[i] / dl; E[i] = lights[l].rgb[i]; }
                } else {
                    const double vv[3] = { lights[l].vec[0] - x[0], lights[l].vec[1] - x[1], lights[l].vec[2] - x[2] };
                    const double d2 = vv[0] * vv[0] + vv[1] * vv[1] + vv[2] * vv[2];
                    const double dl = sqrt(d2);
                    for (int i = 0; i < 3; ++i) wi[i] = vv[i] / dl;
                    const double en[3] = { lights[l].emit_n[0], lights[l].emit_n[1], lights[l].emit_n[2] };
                    double fac = 1.0;
                    if (en[0] != 0.0 || en[1] != 0.0 || en[2] != 0.0) {
                        const double c = -(wi[0] * en[0] + wi[1] * en[1] + wi[2] * en[2]);
                        fac = c > 0.0 ? c : 0.0;
                    }
                    for (int i = 0; i < 3; ++i) E[i] = lights[l].rgb[i] * fac / d2;
                }
                double wi_loc[3], comp[4], rgb[3];
                oracle_to_local(nn, tt, wi, wi_loc);
                pd_components(d, W, b, Z, m, u, v, size, wi_loc, wo_loc, scratch, comp);
                pd_combine(albedo_px ? albedo_px + 12 * (size_t)p : albedos + 12 * (size_t)m, comp, rgb);
                const double c = fabs(wi_loc[2]);
                for (int i = 0; i < 3; ++i) Lp[i] += rgb[i] * E[i] * c;
            }
        }
        free(scratch);
    }
    return 0;
}

int oracle_pd_shade_frame(const oracle_pd_dims* d, const float* const W[7], const float* const b[7], const float* Z,
                          const float* albedos, const float* pos_fp, const float* nrm_u, const float* tan_v,
                          const int32_t* material, int64_t first, int64_t count, const float cam_pos[3],
                          const oracle_pd_light* lights, int n_lights, double* out, int n_threads)
{
    return oracle_pd_shade_frame_px(d, W, b, Z, albedos, NULL, pos_fp, nrm_u, tan_v, material, first, count, cam_pos, lights,
                                    n_lights, out, n_threads);
}

/* Latent interpolation / extrapolation (sec. 6.3): z = (1 - t) z_a + t z_b, t any real ("the material
 * latent vector at 0.9 is computed by extrapolation").  Plain definition in double. */
void oracle_lerp_latent(const float* za, const float* zb, int L, double t, double* out)
{
    for (int i = 0; i < L; ++i) out[i] = (1.0 - t) * (double)za[i] + t * (double)zb[i];
}
