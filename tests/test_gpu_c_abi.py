"""The boundary from C: tests/c/c_abi_smoke.c is compiled with gcc against include/nbsdf.h, linked with libnbsdf.so, the CUDA
runtime and (for the expected values only) liboracle.so, and run on the GPU -- no Python and no torch on that path.
Also: nbsdf_eval inside a captured CUDA graph, and two contexts driven concurrently on two streams.  -m gpu."""
import os
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import oracle.binding  # noqa: E402
from paper_2406_17782_b200 import api, buildlib, synth  # noqa: E402

from test_gpu_parity import check  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_program_through_the_c_abi(tmp_path):
    lib = buildlib.build()
    olib = oracle.binding.build()
    exe = str(tmp_path / "c_abi_smoke")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    subprocess.check_call(["gcc", "-O1", "-std=c11", "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(cuda, "include"),
                           os.path.join(ROOT, "tests", "c", "c_abi_smoke.c"), "-o", exe, lib, olib,
                           "-L" + os.path.join(cuda, "lib64"), "-lcudart", "-lm",
                           "-Wl,-rpath," + os.path.dirname(lib), "-Wl,-rpath," + os.path.dirname(olib),
                           "-Wl,-rpath," + os.path.join(cuda, "lib64")])
    p = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    print(p.stdout.strip())
    assert p.returncode == 0 and p.stdout.startswith("OK"), p.stdout + p.stderr


def test_eval_inside_a_cuda_graph_and_latent_edit_between_replays():
    cfg = synth.config(1, n=70000)
    ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], 16, 64, 8, "fp16")
    api.nbsdf_set_latents(ctx, 0, cfg["latents"])
    n = len(cfg["queries"])
    qd = api.queries_to_device(cfg["queries"])
    out = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        api.nbsdf_eval(ctx, qd, None, n, out)                     # warm-up outside the capture
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for _ in range(3):
            api.nbsdf_eval(ctx, qd, None, n, out)
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"])
    check(out.cpu().numpy(), ref, "fp16", "graph replay")
    Z2 = cfg["latents"].copy()
    Z2[5] = 0.25
    api.nbsdf_set_latents(ctx, 5, Z2[5])                          # an edit between replays is seen by the next replay
    g.replay()
    torch.cuda.synchronize()
    check(out.cpu().numpy(), oracle.eval_queries(cfg["weights"], cfg["biases"], Z2, cfg["queries"]), "fp16", "replay after edit")
    api.nbsdf_destroy(ctx)


def test_host_edits_are_refused_on_a_capturing_stream():
    """include/nbsdf.h: the pinned staging ring cannot be replayed, so set_latents / set_albedos / encode_latent return
    NBSDF_E_INVALID while the stream is being captured and enqueue nothing; the capture itself stays valid."""
    cfg = synth.config(1, n=4096)
    enc = synth.enc_config(feat_width=32, hidden=64, latent=16)
    ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], 16, 64, 8, "fp16")
    api.nbsdf_set_latents(ctx, 0, cfg["latents"])
    api.nbsdf_set_encoder(ctx, enc["weights"], enc["biases"])
    pd = synth.pd_config("eval", n=8)
    pctx = api.nbsdf_create_paper(pd["weights"], pd["biases"], 64, 8, "fp16")
    n = len(cfg["queries"])
    qd = api.queries_to_device(cfg["queries"])
    out = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        api.nbsdf_eval(ctx, qd, None, n, out)
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        for call in (lambda: api.nbsdf_set_latents(ctx, 2, np.full(16, 9.0, np.float32)),
                     lambda: api.nbsdf_encode_latent(ctx, 2, enc["features"][0], 0.5, 1.0),
                     lambda: api.nbsdf_set_albedos(pctx, 0, pd["albedos"])):
            with pytest.raises(api.NbsdfError) as e:
                call()
            assert e.value.status == api.NBSDF_E_INVALID and "captured" in str(e.value)
        api.nbsdf_eval(ctx, qd, None, n, out)
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"])     # row 2 was NOT edited
    check(out.cpu().numpy(), ref, "fp16", "replay after refused edits")
    api.nbsdf_set_latents(ctx, 2, cfg["latents"][2])                                                # and works again outside
    torch.cuda.synchronize()
    api.nbsdf_destroy(ctx)
    api.nbsdf_destroy(pctx)


def test_two_contexts_on_two_streams_concurrently():
    ca, cb = synth.config(1, n=200000), synth.config(4, n=150000, L=32, H=128, seed=77)
    xa = api.nbsdf_create(ca["weights"], ca["biases"], 16, 64, 8, "fp16")
    xb = api.nbsdf_create(cb["weights"], cb["biases"], 32, 128, 8, "fp16")
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    api.nbsdf_set_latents(xa, 0, ca["latents"], stream=sa.cuda_stream)
    api.nbsdf_set_latents(xb, 0, cb["latents"], stream=sb.cuda_stream)
    qa, qb = api.queries_to_device(ca["queries"]), api.queries_to_device(cb["queries"])
    oa = torch.empty((len(ca["queries"]), 3), dtype=torch.float32, device="cuda")
    ob = torch.empty((len(cb["queries"]), 3), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    for _ in range(5):                                            # interleaved launches; the kernels overlap or queue, either is fine
        api.nbsdf_eval(xa, qa, None, len(ca["queries"]), oa, stream=sa.cuda_stream)
        api.nbsdf_eval(xb, qb, None, len(cb["queries"]), ob, stream=sb.cuda_stream)
    torch.cuda.synchronize()
    check(oa.cpu().numpy(), oracle.eval_queries(ca["weights"], ca["biases"], ca["latents"], ca["queries"]), "fp16", "stream a")
    check(ob.cpu().numpy(), oracle.eval_queries(cb["weights"], cb["biases"], cb["latents"], cb["queries"]), "fp16", "stream b")
    api.nbsdf_destroy(xa)
    api.nbsdf_destroy(xb)
