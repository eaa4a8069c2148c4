"""CPU-only checks of the host side: the C-ABI library builds, loads and exports every symbol include/nbsdf.h
declares; the binding validates shapes; no compute call is made (there is no GPU here, and no CPU fallback)."""
import os
import re

import numpy as np
import pytest

from paper_2406_17782_b200 import api, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol(built_lib):
    header = open(os.path.join(ROOT, "include", "nbsdf.h")).read()
    declared = set(re.findall(r"\b(nbsdf_[a-z_]+)\s*\(", header))
    assert declared == set(api.EXPORTS)
    lib = api.load()
    for name in declared:
        assert hasattr(lib, name), name


def test_binding_validates_shapes_before_calling_the_library():
    c = synth.config(0, n=4)
    bad = [w.copy() for w in c["weights"]]
    bad[3] = bad[3][:, :-1]
    with pytest.raises(ValueError):
        api.nbsdf_create(bad, c["biases"], 16, 64, 1)


def test_create_fails_loudly_without_a_gpu_or_returns_a_context():
    import torch
    c = synth.config(0, n=4)
    if torch.cuda.is_available():
        pytest.skip("GPU present: covered by the gpu tests")
    with pytest.raises(api.NbsdfError):
        api.nbsdf_create(c["weights"], c["biases"], 16, 64, 1)


def test_wire_formats_match_the_header():
    assert synth.QUERY_DTYPE.itemsize == 40 and synth.LIGHT_DTYPE.itemsize == 40
    assert [synth.QUERY_DTYPE.fields[k][1] for k in ("u", "v", "footprint", "material", "wi", "wo")] == [0, 4, 8, 12, 16, 28]
    assert [synth.LIGHT_DTYPE.fields[k][1] for k in ("type", "vec", "rgb", "emit_n")] == [0, 4, 16, 28]
    import ctypes as C
    assert C.sizeof(api._GBuffer) == 4 * 8 + 8 + 12 + 4 + 8   # 4 pointers, w, h, cam[3], padding to 8, albedo pointer
