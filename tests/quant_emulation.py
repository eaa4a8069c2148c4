#!/usr/bin/env python
"""TEST INFRASTRUCTURE, NOT PRODUCT CODE -- accuracy study of reduced-precision operands.

PAPER.md:271-273 (sec. 6.4): "other techniques could be used to accelerate its speed further".  The candidate is FP8
(e4m3) operands on the tensor cores (kind::f8f6f4 doubles the dense tensor peak).  This script answers the accuracy half
of that question WITHOUT any GPU code: a numpy fp64 forward pass of the BASELINE.json decoder, layer by layer exactly as
oracle/nbsdf_oracle.c defines it, with a rounding hook on every tensor-core operand --
the inputs x = [z, u', v', lf], y-tail = [wi, wo], the hidden activations h1, h2, g1, g2, the feature, and the weights --
while accumulation, biases and the output activation stay exact, as they do in an fp32-accumulate tensor-core kernel.
With identity hooks it must reproduce the C oracle (asserted on every run), so every number it prints is "oracle with
the named operands rounded".  It calls only oracle/ and the seeded input generator.

    python tests/quant_emulation.py [--n 65536] [--md]      # prints the table of BASELINE.md sec. 5

Formats: fp16 (11-bit significand), bf16 (8), e4m3 (4; max 448, subnormals down to 2^-9, saturating) with a per-layer
power-of-two scale chosen from the layer's own max magnitude (the best case for a per-layer-scaled FP8 kernel), e5m2 (3).
"""
import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2406_17782_b200 import synth  # noqa: E402  (seeded inputs only; none of the method's arithmetic)


def round_sig(x, sig_bits, emin, emax_val=None):
    """Round fp64 to a binary format with `sig_bits` significand bits (incl. the hidden one), RNE, gradual underflow
    below 2^emin, saturation at emax_val (None: no overflow handling)."""
    x = np.asarray(x, np.float64)
    m, e = np.frexp(x)                                   # x = m 2^e, 0.5 <= |m| < 1
    e = np.maximum(e, emin + 1)                          # subnormals: fixed quantum 2^(emin - sig_bits + 1)
    q = np.ldexp(1.0, e - sig_bits)
    y = np.rint(x / q) * q                               # rint = round half to even
    if emax_val is not None:
        y = np.clip(y, -emax_val, emax_val)
    return y


def fp16(x):
    return round_sig(x, 11, -14, 65504.0)


def bf16(x):
    return round_sig(x, 8, -126)


def e4m3_raw(x):
    return round_sig(x, 4, -6, 448.0)


def e5m2_raw(x):
    return round_sig(x, 3, -14, 57344.0)


def scaled(fmt_raw, fmt_max):
    """per-tensor power-of-two scale so that max|x| lands just below the format's maximum"""
    def f(x):
        a = float(np.max(np.abs(x))) if np.size(x) else 0.0
        if a == 0.0:
            return np.asarray(x, np.float64)
        s = 2.0 ** np.floor(np.log2(fmt_max / a))
        return fmt_raw(np.asarray(x, np.float64) * s) / s
    return f


e4m3 = scaled(e4m3_raw, 448.0)
e5m2 = scaled(e5m2_raw, 57344.0)
ident = lambda x: np.asarray(x, np.float64)          # noqa: E731


def forward(cfg, q, r_in=ident, r_act=ident, r_w=ident, r_last=None, merged=False):
    """SURVEY.md sec. 8(c) steps 2-7 in fp64 with operand rounding hooks.  r_in: inputs of layers 1 and 4 (x and the
    [wi, wo] tail); r_act: hidden activations and the feature; r_w: weights; r_last: g2 (default r_act).
    merged: layers 3+4 multiplied out in fp64 before the weight rounding (what nbsdf_eval does for H <= 64), so the
    feature is never rounded."""
    W = [np.asarray(w, np.float64) for w in cfg["weights"]]
    b = [np.asarray(x, np.float64) for x in cfg["biases"]]
    Z = np.asarray(cfg["latents"], np.float64)
    r_last = r_act if r_last is None else r_last
    F = W[2].shape[0]
    u = q["u"].astype(np.float64)
    v = q["v"].astype(np.float64)
    up, vp = u - np.floor(u), v - np.floor(v)
    lf = np.log2(np.minimum(np.maximum(q["footprint"].astype(np.float64), 2.0 ** -20), 16.0))
    x = np.concatenate([Z[q["material"]], up[:, None], vp[:, None], lf[:, None]], axis=1)
    tail = np.concatenate([q["wi"].astype(np.float64), q["wo"].astype(np.float64)], axis=1)
    h1 = np.maximum(r_in(x) @ r_w(W[0]).T + b[0], 0.0)
    h2 = np.maximum(r_act(h1) @ r_w(W[1]).T + b[1], 0.0)
    if merged:
        W34 = W[3][:, :F] @ W[2]
        b34 = W[3][:, :F] @ b[2] + b[3]
        g1 = np.maximum(r_act(h2) @ r_w(W34).T + r_in(tail) @ r_w(W[3][:, F:]).T + b34, 0.0)
    else:
        feat = r_act(h2) @ r_w(W[2]).T + b[2]
        g1 = np.maximum(r_act(feat) @ r_w(W[3][:, :F]).T + r_in(tail) @ r_w(W[3][:, F:]).T + b[3], 0.0)
    g2 = np.maximum(r_act(g1) @ r_w(W[4]).T + b[4], 0.0)
    o = r_last(g2) @ r_w(W[5]).T + b[5]
    return np.where(o > 0, o + np.log1p(np.exp(-np.abs(o))), np.log1p(np.exp(-np.abs(o))))


def rel(a, ref):
    r = np.abs(a - ref) / np.maximum(np.abs(ref), 1e-6)
    return float(r.max()), float(r.mean())


VARIANTS = [
    # name, r_in, r_act, r_w
    ("fp16 operands (shipped default)", fp16, fp16, fp16),
    ("bf16 operands (shipped)", bf16, bf16, bf16),
    ("e4m3 hidden activations only; inputs + weights fp16 (not expressible in one tcgen05 kind)", fp16, e4m3, fp16),
    ("e4m3 activations AND weights, per-layer scales; inputs fp16 (kind::f8f6f4 needs both 8-bit)", fp16, e4m3, e4m3),
    ("e4m3 everything incl. inputs", e4m3, e4m3, e4m3),
    ("e5m2 activations, e4m3 weights", fp16, e5m2, e4m3),
]
POINTS = [("configs[1]  L=16 H=64", 16, 64, 1), ("sweep point L=16 H=128", 16, 128, synth.sweep_seed(1, 2, 1)),
          ("sweep point L=32 H=64", 32, 64, synth.sweep_seed(1, 1, 2))]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=1 << 16)
    ap.add_argument("--md", action="store_true")
    args = ap.parse_args()
    rows = []
    for name, L, H, seed in POINTS:
        cfg = synth.config(4 if seed != 1 else 1, n=args.n, L=L, H=H, seed=seed)
        q = cfg["queries"]
        ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], q)
        self_check = rel(forward(cfg, q), ref)[0]
        assert self_check < 1e-12, self_check               # identity hooks == the C oracle
        assert rel(forward(cfg, q, merged=True), ref)[0] < 1e-12
        for vname, r_in, r_act, r_w in VARIANTS:
            mx, mean = rel(forward(cfg, q, r_in, r_act, r_w, merged=H <= 64), ref)
            rows.append((name, vname, mx, mean))
    if args.md:
        print(f"| point ({args.n} queries) | operands | max rel | mean rel | vs bound (1e-2 / 2e-3) |")
        print("|---|---|---|---|---|")
        for name, vname, mx, mean in rows:
            print(f"| {name} | {vname} | {mx:.2e} | {mean:.2e} | {mx / 1e-2:.1f}x / {mean / 2e-3:.1f}x |")
    else:
        for name, vname, mx, mean in rows:
            print(f"{name:26s} {vname:88s} max {mx:.3e}  mean {mean:.3e}")


if __name__ == "__main__":
    main()
