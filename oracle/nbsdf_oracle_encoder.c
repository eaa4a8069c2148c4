/*
 * nbsdf_oracle_encoder.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain fp64 CPU definition of the ENCODER TAIL: the fully connected residual block that
 * turns a pre-computed ResNet feature of the fabric pattern plus the appearance parameters into the material latent
 * vector.  Same rules as the other oracle files: only tests/, smoke() and bench.py's CPU legs may call it; it shares
 * nothing with the CUDA library.
 *
 * Passages followed (PAPER.md line / section):
 *   "we feed the feature together with the appearance parameters into a residual block, which consists of two fully
 *    connected layers of size 128, and output a material latent vector of size 64"       PAPER.md:162 (sec. 4.2 "Encoder")
 *   "Both the encoder and decoder include a residual block composed of two fully connected layers and a skip
 *    connection before the last leaky ReLU function."                                    PAPER.md:168 (Fig. 3 caption)
 *   appearance parameters = roughness alpha and height-field scaling beta                PAPER.md:168, Table 1 (73-80)
 *   used when a material is initialised or edited, "costs about 0.5 ms"
 *
 * What it computes, in this order (x = [feature(0..Fr), alpha, beta]):
 *   e0 = lrelu(E0 x  + b0)               input projection  (Fr + 2) -> He      -- needed for the skip to have a width
 *   r  = lrelu(E1 e0 + b1)               residual block, first fully connected layer   He -> He
 *   e2 = lrelu(E2 r  + b2 + e0)          second one; the skip is added BEFORE the last leaky ReLU
 *   z  = E3 e2 + b3                      linear output     He -> L (latent, 64 in the paper)
 * Readings (the paper gives only the two sentences above; listed in DESIGN.md sec. 12): the ResNet-18 trunk is out of
 * scope (no textures, no weights), so its output enters as a given vector of width Fr; the in / out projections exist
 * because (Fr + 2) != 128 != 64; the skip source is the block's input e0, mirroring the decoder's block
 * (nbsdf_oracle_paper.c step 4); leaky-ReLU slope 0.01 (unstated); the output is linear (a latent, not an activation).
 * Each W x is the naive double loop in index order.
 *
 * Pins: tests/test_oracle_encoder_pins.py.  Agreement with the paper's trained encoder: "parity unpinned" (no weights).
 */
#include <stdint.h>
#include <stdlib.h>

#define ENC_SLOPE 0.01

typedef struct {
    int32_t feat_width;   /* Fr: width of the pre-computed ResNet feature */
    int32_t hidden;       /* He: 128 in the paper */
    int32_t latent_dim;   /* L: 64 in the paper */
} oracle_enc_dims;

static double enc_lrelu(double x) { return x >= 0.0 ? x : ENC_SLOPE * x; }

/* y = W x + b, W row-major [n_out][n_in] fp32 promoted exactly to double */
static void enc_affine(const float* W, const float* b, int n_out, int n_in, const double* x, double* y)
{
    for (int o = 0; o < n_out; ++o) {
        double acc = (double)b[o];
        for (int i = 0; i < n_in; ++i) acc += (double)W[(size_t)o * n_in + i] * x[i];
        y[o] = acc;
    }
}

/* W[4], b[4]: E0 [He][Fr+2], E1 [He][He], E2 [He][He], E3 [L][He]; feature: Fr fp32; z_out: L doubles */
int oracle_encode_latent(const oracle_enc_dims* d, const float* const* W, const float* const* b, const float* feature,
                         double alpha, double beta, double* z_out)
{
    const int Fr = d->feat_width, He = d->hidden, L = d->latent_dim;
    if (Fr < 0 || He < 1 || L < 1) return -1;
    double* x = (double*)malloc(sizeof(double) * (size_t)(Fr + 2 + 3 * He));
    if (!x) return -2;
    double* e0 = x + Fr + 2;
    double* r = e0 + He;
    double* e2 = r + He;
    for (int i = 0; i < Fr; ++i) x[i] = (double)feature[i];
    x[Fr] = alpha;
    x[Fr + 1] = beta;
    enc_affine(W[0], b[0], He, Fr + 2, x, e0);
    for (int i = 0; i < He; ++i) e0[i] = enc_lrelu(e0[i]);
    enc_affine(W[1], b[1], He, He, e0, r);
    for (int i = 0; i < He; ++i) r[i] = enc_lrelu(r[i]);
    enc_affine(W[2], b[2], He, He, r, e2);
    for (int i = 0; i < He; ++i) e2[i] = enc_lrelu(e2[i] + e0[i]);
    enc_affine(W[3], b[3], L, He, e2, z_out);
    free(x);
    return 0;
}
