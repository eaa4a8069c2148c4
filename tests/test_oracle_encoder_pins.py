"""Pins of the encoder-tail oracle (oracle/nbsdf_oracle_encoder.c) against what the paper's two
sentences and plain mathematics fix: hand-computed one-unit networks (incl. the case that tells "skip before the last
leaky ReLU" from its two plausible misreadings), zero weights -> biases, the no-clip case against an independently written
affine composition that includes the skip term, the all-negative chain that pins the slope, and the place of alpha and
beta in the input vector.  CPU only."""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2406_17782_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "encoder_one_unit.json")


def test_hand_computed_one_unit_networks():
    gold = json.load(open(GOLD))
    for c in gold["cases"]:
        W = [np.array(c[k], np.float32) for k in ("E0", "E1", "E2", "E3")]
        b = [np.array(c[k], np.float32) for k in ("b0", "b1", "b2", "b3")]
        z = oracle.encode_latent(W, b, np.array(c["feature"], np.float32), c["alpha"], c["beta"])
        np.testing.assert_allclose(z, c["z"], rtol=0, atol=1e-14, err_msg=c["name"])


def test_zero_weights_give_biases():
    cfg = synth.enc_config(feat_width=40, hidden=16, latent=8, seed=5)
    W, b = [w.copy() for w in cfg["weights"]], cfg["biases"]
    W[3][:] = 0.0                                      # output layer dead: z = b3 whatever the inputs
    z = oracle.encode_latent(W, b, cfg["features"][0], 0.3, 1.2)
    np.testing.assert_array_equal(z, b[3].astype(np.float64))
    W = [w.copy() for w in cfg["weights"]]
    W[0][:] = 0.0                                      # input projection dead: z independent of feature, alpha, beta
    z1 = oracle.encode_latent(W, b, cfg["features"][0], 0.3, 1.2)
    z2 = oracle.encode_latent(W, b, cfg["features"][1], 0.9, 0.1)
    np.testing.assert_array_equal(z1, z2)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_no_clip_case_is_the_affine_composition_with_the_skip_term(seed):
    """all weights, biases and inputs >= 0: no leaky ReLU clips, so z = E3 ((E2 E1 + I) (E0 x + b0) + E2 b1 + b2) + b3 --
    written here with matrices in transposed storage and a different association, in float64 numpy"""
    rng = np.random.default_rng(seed)
    Fr, He, L = 7, 5, 3
    W = [rng.uniform(0, 1, s).astype(np.float32) for s in synth.enc_layer_shapes(Fr, He, L)]
    b = [rng.uniform(0, 1, s[0]).astype(np.float32) for s in synth.enc_layer_shapes(Fr, He, L)]
    f = rng.uniform(0, 1, Fr).astype(np.float32)
    al, be = 0.375, 1.5
    x = np.concatenate([f.astype(np.float64), [al, be]])
    E0t, E1t, E2t, E3t = [w.astype(np.float64).T for w in W]
    e0 = x @ E0t + b[0]
    want = (e0 @ (E1t @ E2t + np.eye(He)) + b[1].astype(np.float64) @ E2t + b[2]) @ E3t + b[3]
    np.testing.assert_allclose(oracle.encode_latent(W, b, f, al, be), want, rtol=1e-13)


def test_all_negative_chain_pins_the_slope_and_its_three_applications():
    """one unit per layer, every pre-activation negative: z = E3 * s*(E2*s*(E1*s*p0 + b1) + b2 + s*p0) + b3, s = 0.01"""
    W = [np.array([[1.0, 0.0, 0.0]], np.float32), np.array([[1.0]], np.float32), np.array([[1.0]], np.float32), np.array([[1.0]], np.float32)]
    b = [np.array([-3.0], np.float32), np.array([-1.0], np.float32), np.array([-2.0], np.float32), np.array([0.0], np.float32)]
    z = oracle.encode_latent(W, b, np.array([1.0], np.float32), 0.0, 0.0)
    p0 = 1.0 - 3.0                                      # -2      -> e0 = -0.02
    r = 0.01 * (0.01 * p0 - 1.0)                        # -0.0102
    want = 0.01 * (r - 2.0 + 0.01 * p0)                 # -0.020302
    np.testing.assert_allclose(z, [want], rtol=1e-14)


def test_alpha_and_beta_are_the_last_two_inputs_in_that_order():
    cfg = synth.enc_config(feat_width=6, hidden=4, latent=2, seed=9)
    W, b = [w.copy() for w in cfg["weights"]], cfg["biases"]
    f = cfg["features"][0]
    base = oracle.encode_latent(W, b, f, 0.2, 0.7)
    W2 = [w.copy() for w in W]
    W2[0][:, 6] = 0.0                                   # column of alpha
    assert np.array_equal(oracle.encode_latent(W2, b, f, 0.2, 0.7), oracle.encode_latent(W2, b, f, 0.9, 0.7))
    assert not np.array_equal(oracle.encode_latent(W2, b, f, 0.2, 0.7), oracle.encode_latent(W2, b, f, 0.2, 0.1))
    W3 = [w.copy() for w in W]
    W3[0][:, 7] = 0.0                                   # column of beta
    assert np.array_equal(oracle.encode_latent(W3, b, f, 0.2, 0.7), oracle.encode_latent(W3, b, f, 0.2, 0.1))
    assert not np.array_equal(base, oracle.encode_latent(W, b, f, 0.21, 0.7))
