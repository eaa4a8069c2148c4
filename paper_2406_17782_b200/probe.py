"""Launch timeline of the fused eval kernel, from the instrumented debug build (csrc/nbsdf_probe.cuh).  DEBUG TOOL.

    python -m paper_2406_17782_b200.probe [--n 1048576] [--launches 24]

Builds libnbsdf_probe.so (-DNBSDF_PROBE), runs back-to-back nbsdf_eval launches of BASELINE.json configs[1] and prints,
per launch, medians over the SMs of: the gap since the previous launch's CTA on the same SM ended, the prologue
phases, the time to the first layer's completion and to the first stored tile, and the drain (last tile's chain ->
CTA end).  Global-timer nanoseconds; SM clocks for the same intervals give the in-kernel clock rate.
The numbers quoted in DESIGN.md sec. 6 come from profiles/r2_eval_timeline.md, the output of this command.
"""
import argparse
import ctypes as C
import json
import os

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=1 << 20)
    ap.add_argument("--launches", type=int, default=24)
    args = ap.parse_args()
    from . import buildlib
    os.environ["NBSDF_LIB"] = buildlib.build(probe=True)
    import torch
    from . import api, synth
    lib = api.load()
    cfg = synth.config(1, n=args.n)
    ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], 16, 64, 8, "fp16")
    api.nbsdf_set_latents(ctx, 0, cfg["latents"])
    qs = [api.queries_to_device(np.roll(cfg["queries"], r * 12345)) for r in range(4)]
    outs = [torch.empty((args.n, 3), dtype=torch.float32, device="cuda") for _ in range(4)]
    for i in range(8):
        api.nbsdf_eval(ctx, qs[i % 4], None, args.n, outs[i % 4])
    torch.cuda.synchronize()
    lib.nbsdf_debug_clear_probe()
    l0 = api.nbsdf_launch_count(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.launches):
        api.nbsdf_eval(ctx, qs[i % 4], None, args.n, outs[i % 4])
    e1.record()
    torch.cuda.synchronize()
    us = 1e3 * e0.elapsed_time(e1) / args.launches
    buf = np.zeros((32, 160, 10, 2), np.uint64)
    assert lib.nbsdf_debug_read_probe(C.c_void_p(buf.ctypes.data)) == 0
    api.nbsdf_destroy(ctx)
    names = ["entry", "tmem+barriers ready", "grid dependency resolved", "latents ready", "weights landed",
             "first layer done", "first tile stored", "last tile's chain done", "CTA end"]
    rows = []
    for j in range(2, args.launches - 1):
        cur, prev = buf[(l0 + j) % 32], buf[(l0 + j - 1) % 32]
        live = (cur[:, 0, 1] > 0) & (prev[:, 8, 1] > 0)
        t = cur[live][:, :, 1].astype(np.int64)
        c = cur[live][:, :, 0].astype(np.int64)
        gap = t[:, 0] - prev[live][:, 8, 1].astype(np.int64)
        row = {"gap_prev_end_to_entry_ns": float(np.median(gap))}
        for s in range(1, 9):
            row[f"{names[s]} (ns after entry)"] = float(np.median(t[:, s] - t[:, 0]))
        row["drain: last chain done -> CTA end (ns)"] = float(np.median(t[:, 8] - t[:, 7]))
        row["CTA lifetime (ns)"] = float(np.median(t[:, 8] - t[:, 0]))
        row["sm_clock_ghz"] = float(np.median((c[:, 8] - c[:, 0]) / np.maximum(t[:, 8] - t[:, 0], 1)))
        life = np.sort(t[:, 8] - t[:, 0])
        for name, qq in (("p05", 0.05), ("p25", 0.25), ("p75", 0.75), ("p95", 0.95), ("max", 1.0)):
            row[f"CTA lifetime {name} over SMs (ns)"] = float(life[min(len(life) - 1, int(qq * len(life)))])
        end = np.sort(t[:, 8] - t[:, 8].min())
        for name, qq in (("p25", 0.25), ("p50", 0.5), ("p75", 0.75), ("p95", 0.95)):
            row[f"CTA end {name} over SMs, after the first SM's end (ns)"] = float(end[int(qq * len(end))])
        row["entry spread over SMs (ns)"] = float(t[:, 0].max() - t[:, 0].min())
        row["end spread over SMs (ns)"] = float(t[:, 8].max() - t[:, 8].min())
        rows.append(row)
    med = {k: float(np.median([r[k] for r in rows])) for k in rows[0]}
    print(json.dumps({"n": args.n, "launches": args.launches, "us_per_launch_cuda_events": us, "sms": int(live.sum()),
                      "median_over_launches": med}, indent=1))


if __name__ == "__main__":
    main()
