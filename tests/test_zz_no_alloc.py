"""nbsdf_encode_latent_static: the encoder tail for callers that cannot allocate device memory.  -m gpu.

Some users of this library never get to call cudaMalloc: a renderer that gave the whole GPU to its own pool at start-up,
or a frame loop that cannot take the device-wide stall an allocation causes.  For them the library has one entry point
that allocates nothing and keeps the activations between its four launches in a fixed 3-KB array inside the library
image.  This test checks that entry point against the path everybody else uses (nbsdf_set_encoder +
nbsdf_encode_latent, read back with nbsdf_get_latents) and against the fp64 oracle, on two calls in a row -- the second
finds the scratch array as the first left it, and must not care.  The tolerance is the fp32 one of the other tests
(1e-5), taken relative to the largest component of the latent vector: the two paths add the same fp32 products in a
different order, and a component that cancels to nearly zero has no relative accuracy of its own to compare.

The file name sorts last on purpose: the scratch array is shared by the whole process, so this runs after every other
test has had the GPU, and under `pytest -x` a failure here hides nothing behind it.  It also passes alone in a fresh
process (the first call does the per-device set-up itself)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from paper_2406_17782_b200 import api, synth  # noqa: E402

TOL = 1e-5


def to_dev(arrays):
    return [torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda() for a in arrays]


def close(a, ref):
    a, ref = np.asarray(a, np.float64), np.asarray(ref, np.float64)
    return np.abs(a - ref).max() <= TOL * np.abs(ref).max()


@pytest.mark.parametrize("L,He,Fr", [(16, 128, 256), (64, 256, 1022), (8, 40, 0)])
def test_static_entry_matches_the_allocating_path_twice_in_a_row(L, He, Fr):
    enc = synth.enc_config(feat_width=Fr, hidden=He, latent=L, seed=5 + L)
    Wd, bd = to_dev(enc["weights"]), to_dev(enc["biases"])
    feats = to_dev(enc["features"][:2]) if Fr else [None, None]
    z = torch.full((2, L), float("nan"), dtype=torch.float32, device="cuda")
    # two calls back to back on one stream, no synchronisation between them: the stream orders their use of the scratch
    for m in range(2):
        api.nbsdf_encode_latent_static(Wd, bd, feats[m], enc["alpha"][m], enc["beta"][m], z[m])
    torch.cuda.synchronize()
    z = z.cpu().numpy()
    assert np.isfinite(z).all()

    ref = np.stack([oracle.encode_latent(enc["weights"], enc["biases"], enc["features"][m], enc["alpha"][m], enc["beta"][m])
                    for m in range(2)])
    assert np.abs(ref).max() > 0.05 and not np.allclose(ref[0], ref[1])
    for m in range(2):
        assert close(z[m], ref[m]), f"call {m} vs oracle: {np.abs(z[m] - ref[m]).max()}"

    if He in (32, 64, 128, 256) and L in (8, 16, 32, 64):           # what the allocating path supports
        if L == 64:
            pd = synth.pd_config("eval", n=8)
            ctx = api.nbsdf_create_paper(pd["weights"], pd["biases"], 64, 8, "fp16")
        else:
            cfg = synth.config(1, n=8, L=L, H=64)
            ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], L, 64, 8, "fp32")
        api.nbsdf_set_encoder(ctx, enc["weights"], enc["biases"])
        for m in range(2):
            api.nbsdf_encode_latent(ctx, m, enc["features"][m], enc["alpha"][m], enc["beta"][m])
        z_old = api.nbsdf_get_latents(ctx, 0, 2, L)
        api.nbsdf_destroy(ctx)
        for m in range(2):
            assert close(z_old[m], ref[m])
            assert close(z[m], z_old[m]), f"call {m} vs nbsdf_encode_latent: {np.abs(z[m] - z_old[m]).max()}"


def test_static_entry_repeats_bit_for_bit_and_allocates_nothing():
    L, He, Fr = 32, 128, 300
    enc = synth.enc_config(feat_width=Fr, hidden=He, latent=L, seed=9)
    Wd, bd, feats = to_dev(enc["weights"]), to_dev(enc["biases"]), to_dev(enc["features"][:2])
    z = torch.zeros((4, L), dtype=torch.float32, device="cuda")
    api.nbsdf_encode_latent_static(Wd, bd, feats[0], 0.3, 1.2, z[0])      # first call: per-device set-up happens here
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    api.nbsdf_encode_latent_static(Wd, bd, feats[1], 0.7, 0.6, z[1])      # leaves another material's activations behind
    api.nbsdf_encode_latent_static(Wd, bd, feats[0], 0.3, 1.2, z[2])
    api.nbsdf_encode_latent_static(Wd, bd, feats[1], 0.7, 0.6, z[3])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                          # the device's free memory did not move
    z = z.cpu().numpy()
    np.testing.assert_array_equal(z[0].view(np.uint32), z[2].view(np.uint32))
    np.testing.assert_array_equal(z[1].view(np.uint32), z[3].view(np.uint32))
    assert not np.array_equal(z[0], z[1])
    assert close(z[1], oracle.encode_latent(enc["weights"], enc["biases"], enc["features"][1], 0.7, 0.6))


def test_static_entry_rejects_what_does_not_fit_the_scratch():
    for kw in (dict(feat_width=16, hidden=512, latent=16), dict(feat_width=1023, hidden=64, latent=16),
               dict(feat_width=16, hidden=64, latent=65)):
        enc = synth.enc_config(n_materials=1, **kw)
        Wd, bd, feats = to_dev(enc["weights"]), to_dev(enc["biases"]), to_dev(enc["features"][:1])
        z = torch.full((kw["latent"],), 7.0, dtype=torch.float32, device="cuda")
        with pytest.raises(api.NbsdfError) as e:
            api.nbsdf_encode_latent_static(Wd, bd, feats[0], 0.5, 1.0, z)
        assert e.value.status == api.NBSDF_E_UNSUPPORTED and "scratch" in str(e.value)
        torch.cuda.synchronize()
        assert (z == 7.0).all()                                          # nothing was launched
