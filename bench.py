#!/usr/bin/env python
"""bench.py -- headline measurement of the nbsdf hot path on B200.

A step is one pass of the fused decoder (stages A1-A4, B1-B7: `nbsdf_eval`) over one batch of BASELINE.json
configs[1]: 2^20 synthetic queries, 8 materials, L=16, H=64, weights stored in bf16, fp32 I/O.  `value` is whole-job
decoder BSDF queries/s with inputs resident in HBM; `e2e` is the same metric through the same C-ABI call with HOST
buffers (pinned host -> device copy of the batch and device -> host read of the result inside the timed region).
The same JSON line also carries the other half of BASELINE.json's metric, the 1920x1080 five-light frame time
(`nbsdf_shade_frame`, stages C1-C3 on configs[2]), timed the same way in its own loop, and the secondary workloads
(4K / 16 lights, per-query frames, the paper-structured decoder, the fp32 CUDA-core variant).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--precision fp16|bf16|fp32] [--impl ours|reference]
    python bench.py --case NAME [--steps K]      # ONE named workload only (what the ncu captures in profiles/ run)
    python bench.py --sweep                      # BASELINE.json configs[4]

Under torchrun (N > 1) every rank processes its own batch (weak scaling, no data-path collective) and the time is
the max over ranks; `--gpus N` without a torchrun environment re-executes itself under torch.distributed.run with N
ranks.  The timed region is R rounds of exactly K launches, each round bracketed by barrier + synchronize; the line
reports the MEDIAN round (and min / max).  `--impl reference` times the fp64 oracle (oracle/, as it stands) on the
host cores.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_MLP_A = 2 * (19 * 64 + 64 * 64 + 64 * 32)                                          # 14 720
FLOP_MLP_B = 2 * (38 * 64 + 64 * 64 + 64 * 3)                                           # 13 440
FLOP_PER_QUERY = FLOP_MLP_A + FLOP_MLP_B                                                # 28 160, unpadded
PD_FLOP_FUSION = 2 * (88 * 64 + 64 * 32)                                                # 15 360
PD_FLOP_ANGULAR = 2 * (37 * 64 + 3 * 64 * 64 + 64 * 4)                                  # 29 824
PD_FLOP_PER_QUERY = PD_FLOP_FUSION + PD_FLOP_ANGULAR                                    # 45 184, unpadded
BYTES_PER_QUERY = 40 + 12
N_ROTATE = 8            # distinct resident batches cycled through so that no step finds its input in L2
ROUNDS = 7              # timed rounds of `steps` launches; the median round is reported
WORKLOAD = "configs[1]: batch eval, 2^20 queries/step/GPU, 8 materials, L=16, H=64, F=32, bf16-stored weights, fp32 I/O"
METRIC = "decoder_bsdf_queries_per_sec"
UNIT = "queries/s"
# fp32 CUDA-core variant: "alu" roofline = 148 SMs x 128 FMA lanes x 2 FLOP x SM clock (guide: 148 SMs, 4 x 32 fp32
# lanes per SM, clocks.max.sm 1965 MHz) = 74.4 TFLOP/s
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def flop_per_query(L, H):
    return 2 * ((L + 3) * H + H * H + H * 32 + 38 * H + H * H + 3 * H)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"bf16_tflops": float(d["bf16_tflops"]), "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", 0)),
                "hbm_gbs": float(d["hbm_gbs"]), "source": "measured"}
    return {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0, "source": "fallback"}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML every few ms while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz, self._stop, self._t = [], set(), None, threading.Event(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _reasons(self):
        nv = self.nv
        try:
            mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            try:
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            except Exception:
                return []
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}
        return [v for k, v in names.items() if mask & k]

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                self.reasons.update(self._reasons())
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()

    def stop(self):
        self._stop.set()
        if self._t is not None:
            self._t.join()
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_rate(cfg, n_sample, threads=0, min_seconds=0.0):
    """queries/s of the fp64 oracle, as it stands, on the first n_sample queries of cfg; the pass is repeated until
    min_seconds of CPU work have been timed.  Returns (rate, seconds, passes)."""
    import oracle
    q = cfg["queries"][:n_sample]
    t0 = time.perf_counter()
    passes = 0
    while True:
        oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], q, n_threads=threads)
        passes += 1
        dt = time.perf_counter() - t0
        if dt >= min_seconds:
            return passes * len(q) / dt, dt, passes


def arm_config(n_step, prec, bounded=False):
    """The `config` of BOTH arms of the bench (the driver compares them): same keys, same values for the same workload."""
    return {"workload": WORKLOAD + (" (bounded sample per step)" if bounded else ""), "queries_per_step_per_gpu": n_step,
            "latent_dim": 16, "hidden": 64, "materials": 8,
            "precision": f"product arm: {prec} operands, fp32 accumulate; reference arm: the fp64 oracle"}


def run_reference(args):
    """--impl reference: the oracle on the host cores, stepping over configs[1].  A step is the FULL 2^20-query batch
    when steps + warmup such steps fit the time budget (they do at the driver's 20 + 3), else a bounded sample of it."""
    from paper_2406_17782_b200 import dist, synth
    rank, _, world = dist.env_world()
    if rank != 0:
        return
    import oracle
    cores = len(os.sched_getaffinity(0))
    n_full = 1 << 20
    cfg = synth.config(1, n=n_full)
    rate0, _, _ = oracle_rate(cfg, 1 << 14)
    budget_s = 150.0
    n_step = int(min(n_full, max(256, rate0 * budget_s / max(1, args.steps + args.warmup))))
    if n_step > 0.9 * n_full:
        n_step = n_full
    for _ in range(args.warmup):
        oracle_rate(cfg, n_step)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"][:n_step])
    dt = time.perf_counter() - t0
    value = n_step * args.steps / dt
    what = "all" if n_step == n_full else f"first {n_step} of the"
    sample = f"{what} 2^20 queries of configs[1] per step, fp64, OpenMP over queries"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": arm_config(n_step, args.precision, bounded=n_step != n_full),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": min(cores, oracle.max_threads()), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def time_loop(torch, fn, steps, barrier):
    """barrier + sync, K calls of fn(i) timed with CUDA events on the current stream, sync + barrier.  Returns ms."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record()
    for i in range(steps):
        fn(i)
    e1.record()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def time_rounds(torch, fn, steps, barrier=lambda: None, reduce_max=lambda ms: ms, rounds=ROUNDS):
    """R rounds of exactly `steps` launches (each round timed as time_loop does, max over ranks): a 20-step run of a
    30-us kernel is otherwise ONE 0.6-ms sample.  Returns (median, min, max) of the per-round milliseconds."""
    ms = sorted(reduce_max(time_loop(torch, fn, steps, barrier)) for _ in range(rounds))
    return ms[len(ms) // 2], ms[0], ms[-1]


# ---------------------------------------------------------------------------------------------------------------------
# Workloads.  Each builder makes the resident device buffers and returns a dict with `step(i)` (one launch), the
# algorithmic work of one launch (`units`, `flop`, `bytes`), the roofline that binds it and `close()`.
def _rotations(arr, n_rot, shift):
    return [np.roll(arr, r * shift, axis=0) for r in range(n_rot)]


def wl_eval(torch, api, synth, dev, prec, L=16, H=64, n=1 << 20, seed=None, frames=False, cfg_idx=1, M=8, order=None):
    """order: None = material ids as the generator draws them (i.i.d. uniform per query: fully incoherent), "sorted" = the
    same queries stably sorted by material id (what a sort/bin pre-pass would hand the kernel)."""
    cfg = synth.config(cfg_idx, n=n, L=L, H=H, seed=seed)
    if M != 8:                                      # the largest gather: a 64-row latent table, ids over the whole range
        rng = np.random.default_rng(1000 + M)
        cfg["latents"] = synth.make_latents(rng, M, L)
        cfg["queries"]["material"] = rng.integers(0, M, size=n).astype(np.int32)
    if order == "sorted":
        cfg["queries"] = cfg["queries"][np.argsort(cfg["queries"]["material"], kind="stable")]
    ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], L, H, M, prec, device=dev.index or 0)
    api.nbsdf_set_latents(ctx, 0, cfg["latents"])
    per_q = BYTES_PER_QUERY + (24 if frames else 0)
    n_rot = N_ROTATE if n * per_q * N_ROTATE <= 3e9 else max(1, int(3e9 // (n * per_q)))
    shift = 12345 if order is None else 0           # a rotation would split the sorted runs; distinct buffers still rotate
    qs = [torch.from_numpy(q.view(np.uint8).reshape(-1).copy()).to(dev) for q in _rotations(cfg["queries"], n_rot, shift)]
    frs = None
    if frames:
        fr_host = synth.make_frames(np.random.default_rng(77), n)
        frs = [torch.from_numpy(f.copy()).to(dev) for f in _rotations(fr_host, n_rot, 12345)]
    outs = [torch.empty((n, 3), dtype=torch.float32, device=dev) for _ in range(n_rot)]

    def step(i):
        api.nbsdf_eval(ctx, qs[i % n_rot], frs[i % n_rot] if frs else None, n, outs[i % n_rot])

    flop = flop_per_query(L, H)
    return {"step": step, "ctx": ctx, "cfg": cfg, "units": n, "flop": flop * n, "bytes": per_q * n, "flop_per_unit": flop,
            "bound": "alu" if prec == "fp32" else "tensor", "q_dev": qs, "out_dev": outs, "n_rot": n_rot,
            "kernel": "eval_fp32_kernel" if prec == "fp32" else f"tc_kernel<{L},{H},{prec},eval>",
            "workload": f"batch eval, {n} queries/launch, {M} materials, L={L}, H={H}, F=32, bf16-stored weights, fp32 I/O"
                        + (", per-query world frame (64 B in + 12 B out)" if frames else "")
                        + (", queries sorted by material id" if order == "sorted" else ""),
            "close": lambda: api.nbsdf_destroy(ctx)}


def wl_frame(torch, api, synth, dev, prec, idx=2, seed=None):
    cfg = synth.config(idx, seed=seed)
    ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], 16, 64, 8, prec, device=dev.index or 0)
    api.nbsdf_set_latents(ctx, 0, cfg["latents"])
    g = cfg["gbuffer"]
    npx = g["width"] * g["height"]
    n_rot = 3 if idx == 2 else 1                     # 1080p: 3 x (108 + 25) MB > L2; 4K: 431 MB of G-buffer > L2
    gds, rads = [], []
    for r in range(n_rot):
        gr = {k: np.roll(g[k], r * 4099, axis=0) for k in ("pos_fp", "nrm_u", "tan_v", "material")}
        gr.update(width=g["width"], height=g["height"], cam_pos=g["cam_pos"])
        gds.append(api.gbuffer_to_device(gr, dev))
        rads.append(torch.empty((npx, 3), dtype=torch.float32, device=dev))
    lights = cfg["lights"]

    def step(i):
        api.nbsdf_shade_frame(ctx, gds[i % n_rot], lights, rads[i % n_rot])

    fpp = FLOP_MLP_A + len(lights) * FLOP_MLP_B
    return {"step": step, "ctx": ctx, "cfg": cfg, "units": npx, "flop": fpp * npx, "bytes": 64 * npx, "flop_per_unit": fpp,
            "bound": "alu" if prec == "fp32" else "tensor", "n_lights": len(lights),
            "kernel": "shade_fp32_kernel" if prec == "fp32" else f"tc_kernel<16,64,{prec},shade>",
            "workload": f"configs[{idx}]: {g['width']}x{g['height']}, 8 materials in 64px tiles, {len(lights)} lights "
                        + ("(1 directional + 4 point)" if idx == 2 else "(4x4 stratified samples of one emitter)"),
            "close": lambda: api.nbsdf_destroy(ctx)}


def wl_paper(torch, api, synth, dev, kind, seed_shift=0):
    """the paper-structured decoder (nbsdf_create_paper), fp16 operands."""
    if kind == "eval":
        n = 1 << 20
        cfg = synth.pd_config("eval", n=n, seed=11 + seed_shift)
    else:
        cfg = synth.pd_config("frame", seed=12 + seed_shift)
    ctx = api.nbsdf_create_paper(cfg["weights"], cfg["biases"], 64, 8, "fp16", device=dev.index or 0)
    api.nbsdf_set_latents(ctx, 0, cfg["latents"])
    api.nbsdf_set_albedos(ctx, 0, cfg["albedos"])
    if kind == "eval":
        qs = [torch.from_numpy(q.view(np.uint8).reshape(-1).copy()).to(dev) for q in _rotations(cfg["queries"], N_ROTATE, 12345)]
        outs = [torch.empty((n, 3), dtype=torch.float32, device=dev) for _ in range(N_ROTATE)]
        step = lambda i: api.nbsdf_eval(ctx, qs[i % N_ROTATE], None, n, outs[i % N_ROTATE])      # noqa: E731
        return {"step": step, "ctx": ctx, "cfg": cfg, "units": n, "flop": PD_FLOP_PER_QUERY * n, "bytes": BYTES_PER_QUERY * n,
                "flop_per_unit": PD_FLOP_PER_QUERY, "bound": "tensor", "kernel": "pd_kernel<64,eval>", "q_dev": qs, "out_dev": outs,
                "workload": "paper-structured decoder (latent 64, one-blob 24, 2 fusion + 5 angular layers, H=64, F=32): "
                            "2^20 Table-2 queries per launch", "close": lambda: api.nbsdf_destroy(ctx)}
    g = cfg["gbuffer"]
    npx = g["width"] * g["height"]
    gds, rads = [], []
    for r in range(3):
        gr = {kk: np.roll(g[kk], r * 4099, axis=0) for kk in ("pos_fp", "nrm_u", "tan_v", "material")}
        gr.update(width=g["width"], height=g["height"], cam_pos=g["cam_pos"])
        gds.append(api.gbuffer_to_device(gr, dev))
        rads.append(torch.empty((npx, 3), dtype=torch.float32, device=dev))
    lights = cfg["lights"]
    step = lambda i: api.nbsdf_shade_frame(ctx, gds[i % 3], lights, rads[i % 3])                  # noqa: E731
    fpp = PD_FLOP_FUSION + len(lights) * PD_FLOP_ANGULAR
    return {"step": step, "ctx": ctx, "cfg": cfg, "units": npx, "flop": fpp * npx, "bytes": 64 * npx, "flop_per_unit": fpp,
            "bound": "tensor", "kernel": "pd_kernel<64,shade>", "n_lights": len(lights),
            "workload": "paper-structured decoder: 1920x1080 frame, 5 direct lights + 1 behind the fabric",
            "close": lambda: api.nbsdf_destroy(ctx)}


CASES = {
    # name: (builder kwargs) -- `python bench.py --case NAME` runs exactly one of these; profiles/*.md cite them
    "eval": lambda t, a, s, d, p: wl_eval(t, a, s, d, p),
    "eval_frames": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, frames=True),
    "eval_h32": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=16, H=32, n=1 << 22, seed=s.sweep_seed(5, 0, 1), cfg_idx=4),
    "eval_h128": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=16, H=128, n=1 << 22, seed=s.sweep_seed(5, 2, 1), cfg_idx=4),
    "eval_l32": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=32, H=64, n=1 << 20, seed=s.sweep_seed(4, 1, 2), cfg_idx=4),
    "eval_h32_frames": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=16, H=32, n=1 << 22, seed=s.sweep_seed(5, 0, 1), cfg_idx=4, frames=True),
    "eval_m64_l32": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=32, H=64, n=1 << 20, seed=s.sweep_seed(4, 1, 2), cfg_idx=4, M=64),
    "eval_m64_l32_h32_frames": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=32, H=32, n=1 << 22, seed=s.sweep_seed(5, 0, 2), cfg_idx=4, M=64, frames=True),
    "eval_sorted": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, order="sorted"),
    "eval_m64_l32_sorted": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, L=32, H=64, n=1 << 20, seed=s.sweep_seed(4, 1, 2), cfg_idx=4, M=64, order="sorted"),
    "eval_2p24": lambda t, a, s, d, p: wl_eval(t, a, s, d, p, n=1 << 24),
    "frame": lambda t, a, s, d, p: wl_frame(t, a, s, d, p, 2),
    "frame_4k": lambda t, a, s, d, p: wl_frame(t, a, s, d, p, 3),
    "paper_eval": lambda t, a, s, d, p: wl_paper(t, a, s, d, "eval"),
    "paper_frame": lambda t, a, s, d, p: wl_paper(t, a, s, d, "frame"),
    "fp32_eval": lambda t, a, s, d, p: wl_eval(t, a, s, d, "fp32"),
    "fp32_frame": lambda t, a, s, d, p: wl_frame(t, a, s, d, "fp32", 2),
}


def measure(torch, w, steps, warmup, peaks, barrier=lambda: None, reduce_max=lambda ms: ms, rounds=ROUNDS):
    """warm-up, then `rounds` rounds of exactly `steps` launches; rates from the median round"""
    for i in range(max(3, warmup)):
        w["step"](i)
    torch.cuda.synchronize()
    med, lo, hi = time_rounds(torch, w["step"], steps, barrier, reduce_max, rounds)
    sec = med * 1e-3 / steps
    tf = w["flop"] / sec / 1e12
    peak = ALU_PEAK_TFLOPS if w["bound"] == "alu" else peaks["bf16_tflops"]
    return {"workload": w["workload"], "kernel": w["kernel"], "ms_per_launch": med / steps, "ms_per_launch_min": lo / steps,
            "ms_per_launch_max": hi / steps, "steps": steps, "rounds": rounds, "units_per_s": w["units"] / sec,
            "flop_per_unit": w["flop_per_unit"], "achieved_tflops": tf, "bound": w["bound"], "peak_tflops": peak,
            "frac": tf / peak, "hbm_gbs_algorithmic": w["bytes"] / sec / 1e9,
            "hbm_frac": w["bytes"] / sec / 1e9 / peaks["hbm_gbs"], "bytes_per_unit": w["bytes"] / w["units"]}


def run_case(args):
    import torch
    from paper_2406_17782_b200 import api, synth
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    w = CASES[args.case](torch, api, synth, dev, args.precision)
    r = measure(torch, w, args.steps, args.warmup, measured_peaks(), rounds=args.rounds)
    r["case"] = args.case
    r["precision"] = args.precision
    w["close"]()
    print(json.dumps(r), flush=True)


def paper_decoder_error(torch, api, synth, w, n_check=1 << 16):
    """max / mean relative error of the paper-structured decoder (fp16 operands) against ITS oracle on a strided sample"""
    import oracle
    cfg = w["cfg"]
    idx = np.arange(0, len(cfg["queries"]), max(1, len(cfg["queries"]) // n_check))
    w["step"](0)
    torch.cuda.synchronize()
    got = w["out_dev"][0].cpu().numpy()[idx].astype(np.float64)
    ref = oracle.pd_eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["albedos"], cfg["queries"][idx])
    rel = np.abs(got - ref) / np.maximum(np.abs(ref), 1e-6)
    return {"max_rel": float(rel.max()), "mean_rel": float(rel.mean()), "checked": int(len(idx)),
            "how": "strided sample of the 2^20 queries vs oracle/nbsdf_oracle_paper.c"}


def run_ours(args):
    import torch
    from paper_2406_17782_b200 import api, dist, synth

    rank, local_rank, world = dist.init("nccl")
    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the torchrun environment has WORLD_SIZE={world}")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    peaks = measured_peaks()
    prec = args.precision
    K, W, R = args.steps, max(args.warmup, 3), args.rounds
    barrier = dist.barrier
    rmax = lambda ms: dist.max_over_ranks(ms, dev)        # noqa: E731

    # ---- headline: configs[1], one distinct batch set per rank (weak scaling) ----
    n = 1 << 20
    w = wl_eval(torch, api, synth, dev, prec, seed=dist.rank_seed(1, rank))
    ctx, cfg, q_dev, out_dev = w["ctx"], w["cfg"], w["q_dev"], w["out_dev"]
    for i in range(W):
        w["step"](i)
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    l0 = api.nbsdf_launch_count(ctx)
    sampler.start()
    ms, ms_min, ms_max = time_rounds(torch, w["step"], K, barrier, rmax, R)
    clocks = sampler.stop()
    launches = (api.nbsdf_launch_count(ctx) - l0) // R          # kernels launched per timed round of K steps
    value = world * n * K / (ms * 1e-3)

    # ---- e2e: HOST buffers through the same call; H2D of the batch and D2H of the result inside the timed region ----
    q_host = torch.from_numpy(cfg["queries"].view(np.uint8).reshape(-1).copy()).pin_memory()
    out_host = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    q_stage = torch.empty_like(q_dev[0])
    o_stage = out_dev[0]
    n_chunks = 8                                     # chunked so that H2D, the kernel and D2H of different chunks overlap
    cq = n // n_chunks
    s_in, s_run, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    ev_in = [torch.cuda.Event() for _ in range(n_chunks)]
    ev_run = [torch.cuda.Event() for _ in range(n_chunks)]

    def step_e2e(i):
        cur = torch.cuda.current_stream()
        for st in (s_in, s_run, s_out):
            st.wait_stream(cur)
        for c in range(n_chunks):
            qb, ob = slice(c * cq * 40, (c + 1) * cq * 40), slice(c * cq, (c + 1) * cq)
            with torch.cuda.stream(s_in):
                q_stage[qb].copy_(q_host[qb], non_blocking=True)
                ev_in[c].record(s_in)
            with torch.cuda.stream(s_run):
                s_run.wait_event(ev_in[c])
                api.nbsdf_eval(ctx, q_stage[qb], None, cq, o_stage[ob], stream=s_run.cuda_stream)
                ev_run[c].record(s_run)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_run[c])
                out_host[ob].copy_(o_stage[ob], non_blocking=True)
        cur.wait_stream(s_out)
        cur.wait_stream(s_run)

    k_e2e = max(3, min(K, 50))
    for i in range(3):
        step_e2e(i)
    torch.cuda.synchronize()
    ms_e2e = rmax(time_loop(torch, step_e2e, k_e2e, barrier))
    e2e_value = world * n * k_e2e / (ms_e2e * 1e-3)

    # ---- the other half of the metric: 1080p, 5 lights (configs[2]); every rank shades its own frame ----
    wf = wl_frame(torch, api, synth, dev, prec, 2, seed=dist.rank_seed(2, rank))
    frame = measure(torch, wf, max(3, min(K, 50)), 3, peaks, barrier, rmax, R)      # <= 7 x 50 x 0.18 ms: stays in the burst regime
    frame["frame_ms"] = frame["ms_per_launch"]
    frame["decoder_evals_per_s"] = world * frame["units_per_s"] * wf["n_lights"]
    wf["close"]()
    del wf
    torch.cuda.empty_cache()

    # ---- the headline kernel in the SUSTAINED regime (rank 0): one ~0.25-s round of back-to-back launches, against the
    # sustained cuBLAS peak -- burst over burst above, sustained over sustained here, never mixed ----
    sustained = None
    if rank == 0 and prec != "fp32":
        k_sus = 8000
        smp = ClockSampler(local_rank)
        smp.start()
        ms_sus = sorted(time_loop(torch, w["step"], k_sus, lambda: None) for _ in range(3))[1]
        clk_sus = smp.stop()
        tf_sus = FLOP_PER_QUERY * n * k_sus / (ms_sus * 1e-3) / 1e12
        sustained = {"launches_per_round": k_sus, "rounds": 3, "ms_per_round": ms_sus, "queries_per_s": n * k_sus / (ms_sus * 1e-3),
                     "achieved": tf_sus, "peak": peaks["bf16_tflops_sustained"] or None, "unit": "TFLOP/s",
                     "frac": tf_sus / peaks["bf16_tflops_sustained"] if peaks["bf16_tflops_sustained"] else None, "clocks": clk_sus}

    # ---- secondary workloads, rank 0 only (not part of the scaled value) ----
    extras = {}
    if rank == 0 and prec != "fp32":
        for key, case, k_cap in (("eval_with_frames", "eval_frames", 200), ("eval_sorted_by_material", "eval_sorted", 200),
                                 ("eval_h32_frames", "eval_h32_frames", 50), ("eval_m64_l32", "eval_m64_l32", 200),
                                 ("eval_m64_l32_sorted", "eval_m64_l32_sorted", 200), ("frame_4k", "frame_4k", 10),
                                 ("paper_eval", "paper_eval", 200), ("paper_frame", "paper_frame", 30),
                                 ("fp32_variant", "fp32_eval", 10), ("fp32_variant_frame", "fp32_frame", 3)):
            wx = CASES[case](torch, api, synth, dev, prec)
            extras[key] = measure(torch, wx, max(3, min(K, k_cap)), 3, peaks, rounds=min(R, 5))
            if case == "paper_eval":
                extras[key]["parity"] = paper_decoder_error(torch, api, synth, wx)
            wx["close"]()
            del wx
            torch.cuda.empty_cache()
        for key in ("frame_4k", "paper_frame", "fp32_variant_frame"):
            extras[key]["frame_ms"] = extras[key]["ms_per_launch"]
        for key in ("eval_with_frames", "eval_sorted_by_material", "eval_h32_frames", "eval_m64_l32", "eval_m64_l32_sorted",
                    "paper_eval", "fp32_variant"):
            extras[key]["queries_per_s"] = extras[key]["units_per_s"]

    line = None
    if rank == 0:
        us_per_launch = 1e3 * ms / K
        achieved_tf = FLOP_PER_QUERY * n / (us_per_launch * 1e-6) / 1e12
        traffic = None
        tp = os.path.join(ROOT, "profiles", "traffic.csv")      # dram bytes/launch copied from the ncu --set full summary
        if os.path.exists(tp):
            for ln in open(tp).read().splitlines()[1:]:
                parts = ln.split(",")
                if parts[0] == f"eval_{prec}_dram_bytes_per_launch":
                    traffic = int(parts[1])
        cores = len(os.sched_getaffinity(0))
        n_cpu = 1 << 20
        cpu_rate, cpu_dt, cpu_passes = oracle_rate(cfg, n_cpu, min_seconds=12.0)
        cpu_rate_1t, _, _ = oracle_rate(cfg, 1 << 16, threads=1, min_seconds=2.0)
        import oracle
        peak = peaks["bf16_tflops"] if prec != "fp32" else ALU_PEAK_TFLOPS
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp16": "f16", "bf16": "bf16", "fp32": "f32"}[prec], "data": "synthetic",
            "config": arm_config(n, prec),
            "notes": {"l2": f"inputs rotate over {N_ROTATE} distinct resident batches "
                            f"({N_ROTATE * n * BYTES_PER_QUERY / 1e6:.0f} MB > 126 MB L2), no flush kernel",
                      "parallelism": f"replicated weights, {world} independent query shards",
                      "timing": f"median of {R} rounds of {K} launches each (ms_per_step_min / _max: the fastest / slowest round)"},
            "ms_per_step_min": ms_min / K, "ms_per_step_max": ms_max / K, "rounds": R,
            "roofline": {"bound": "tensor" if prec != "fp32" else "alu", "achieved": achieved_tf,
                         "peak": peak, "unit": "TFLOP/s", "frac": achieved_tf / peak,
                         "traffic": traffic, "peak_source": (peaks["source"] + " burst (cuBLAS bf16 8192^3)") if prec != "fp32"
                         else "148 SMs x 128 FMA lanes x 2 x 1.965 GHz",
                         "frac_of_sustained": achieved_tf / peaks["bf16_tflops_sustained"] if peaks["bf16_tflops_sustained"] and prec != "fp32" else None,
                         "kernel": w["kernel"], "us_per_launch": us_per_launch, "flop_per_query": FLOP_PER_QUERY,
                         "hbm_gbs_algorithmic": BYTES_PER_QUERY * n / (us_per_launch * 1e-6) / 1e9,
                         # the other half of BASELINE.json's metric ("... and 1080p frame ms"), configs[2], same peak
                         "frame_ms": frame["frame_ms"], "frame_ms_min": frame["ms_per_launch_min"],
                         "frame_ms_max": frame["ms_per_launch_max"], "frame_frac": frame["frac"], "frame_kernel": frame["kernel"],
                         "frame_workload": frame["workload"],
                         "sustained": sustained},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(q_host.numel()),
                    "d2h_bytes_per_step": int(out_host.numel() * 4), "steps": k_e2e,
                    "how": f"{n_chunks} chunks per step: pinned H2D, nbsdf_eval and D2H on three streams chained by events"},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "cpu_baseline": {"value": cpu_rate, "unit": UNIT, "cores": min(cores, oracle.max_threads()), "kind": "oracle", "value_1_thread": cpu_rate_1t,
                             "sample": f"all {n_cpu} queries of configs[1], {cpu_passes} passes, fp64, OpenMP over queries, {cpu_dt:.1f} s"},
        }
        line.update(extras)
        line["frame"] = frame                                   # last on the line: a truncated tail still ends with it
    w["close"]()
    dist.finalize()
    if line is not None:
        print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE.json configs[4]: N in 2^12..2^26 (x4 steps) x H in {32,64,128} x L in {8,16,32}, 8 materials, seed per
    point.  One JSON line per point: queries/s, binding roofline and fraction, and oracle parity on a sample that spans
    the WHOLE batch -- a strided sample plus the last 2^12 queries (the ragged tail and the deepest pipeline rounds),
    min(N, 2^16) queries in all.  Not the headline line; `python bench.py --sweep > profiles/...` regenerates the table."""
    import torch
    import oracle
    from paper_2406_17782_b200 import api, synth
    torch.cuda.set_device(0)
    peaks = measured_peaks()
    prec = args.precision
    Ns = [1 << e for e in range(12, 27, 2)]
    if args.sweep_max_log2 < 26:
        Ns = [n for n in Ns if n <= (1 << args.sweep_max_log2)]
    for i_h, H in enumerate((32, 64, 128)):
        for i_l, L in enumerate((8, 16, 32)):
            flop = flop_per_query(L, H)
            t_tensor = flop / (peaks["bf16_tflops"] * 1e12)
            t_hbm = BYTES_PER_QUERY / (peaks["hbm_gbs"] * 1e9)
            bound = "tensor" if t_tensor >= t_hbm else "hbm"
            for i_n, n in enumerate(Ns):
                cfg = synth.config(4, n=n, L=L, H=H, seed=synth.sweep_seed(i_n, i_h, i_l))
                ctx = api.nbsdf_create(cfg["weights"], cfg["biases"], L, H, 8, prec)
                api.nbsdf_set_latents(ctx, 0, cfg["latents"])
                n_rot = max(1, min(8, int(400e6 // (n * BYTES_PER_QUERY)) + 1)) if n * BYTES_PER_QUERY < 200e6 else 1
                qs = [api.queries_to_device(np.roll(cfg["queries"], r * 977)) for r in range(n_rot)]
                outs = [torch.empty((n, 3), dtype=torch.float32, device="cuda") for _ in range(n_rot)]
                api.nbsdf_eval(ctx, qs[0], None, n, outs[0])
                torch.cuda.synchronize()
                m = min(n, 1 << 16)
                if m == n:
                    idx = np.arange(n)
                else:
                    tail = np.arange(n - (1 << 12), n)
                    idx = np.unique(np.concatenate([np.arange(0, n, n // (m - (1 << 12)))[:m - (1 << 12)], tail]))
                ref = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"][idx])
                got = outs[0][torch.from_numpy(idx).cuda()].cpu().numpy().astype(np.float64)
                rel = np.abs(got - ref) / np.maximum(np.abs(ref), 1e-6)
                k = int(max(10, min(2000, 2e9 / (n * 40))))
                for i in range(5):
                    api.nbsdf_eval(ctx, qs[i % n_rot], None, n, outs[i % n_rot])
                ms = time_rounds(torch, lambda i: api.nbsdf_eval(ctx, qs[i % n_rot], None, n, outs[i % n_rot]), k, rounds=3)[0] / k
                qps = n / (ms * 1e-3)
                us_graph = None
                if n < (1 << 16):                    # launch-bound sizes: also replay 20 launches as one CUDA graph
                    try:
                        g = torch.cuda.CUDAGraph()
                        side = torch.cuda.Stream()
                        side.wait_stream(torch.cuda.current_stream())
                        with torch.cuda.stream(side):
                            for i in range(3):
                                api.nbsdf_eval(ctx, qs[0], None, n, outs[0])
                        torch.cuda.current_stream().wait_stream(side)
                        with torch.cuda.graph(g):
                            for i in range(20):
                                api.nbsdf_eval(ctx, qs[i % n_rot], None, n, outs[i % n_rot])
                        g.replay()
                        us_graph = 1e3 * time_loop(torch, lambda i: g.replay(), 50, lambda: None) / (50 * 20)
                    except Exception as exc:          # capture unsupported: report the stream figure only
                        us_graph = f"unavailable: {type(exc).__name__}"
                frac = qps * (t_tensor if bound == "tensor" else t_hbm)
                print(json.dumps({"config": 4, "n": n, "H": H, "L": L, "precision": prec, "us_per_launch": ms * 1e3,
                                  "us_per_launch_cuda_graph": us_graph, "queries_per_s": qps, "flop_per_query": flop, "bound": bound, "roofline_frac": frac,
                                  "tensor_frac": qps * t_tensor, "hbm_frac": qps * t_hbm, "launches_timed": k,
                                  "rotating_batches": n_rot, "parity_queries": int(len(idx)),
                                  "parity_sample": "all" if m == n else "strided over the whole batch + the last 4096",
                                  "max_rel": float(rel.max()), "mean_rel": float(rel.mean())}), flush=True)
                api.nbsdf_destroy(ctx)
                del qs, outs
                torch.cuda.empty_cache()


def run_plumbing_check(args):
    """The rank plumbing of run_ours without a GPU (gloo): rendezvous, --gpus == WORLD_SIZE, barrier-bracketed timing
    reduced with max over ranks, one line from rank 0.  What tests/test_bench_plumbing.py launches with --gpus 2."""
    from paper_2406_17782_b200 import dist
    rank, local_rank, world = dist.init("gloo")
    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the torchrun environment has WORLD_SIZE={world}")
    dist.barrier()
    ms = dist.max_over_ranks(10.0 + rank)
    seen = dist.sum_over_ranks(1.0)
    dist.barrier()
    dist.finalize()
    if rank == 0:
        print(json.dumps({"plumbing_check": True, "n_gpus": world, "ranks_seen": int(seen), "max_over_ranks_ms": ms,
                          "seeds": [dist.rank_seed(1, r) for r in range(world)]}), flush=True)


def respawn_under_torchrun(args):
    """`--gpus N` (N > 1) launched plainly: re-execute this command line under torch.distributed.run with N ranks on this
    node (rendezvous on 127.0.0.1), so that the documented entry point produces the N-rank line by itself."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--rounds", type=int, default=ROUNDS, help="timed rounds of --steps launches; the median is reported")
    ap.add_argument("--precision", default="fp16", choices=["fp16", "bf16", "fp32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--case", default=None, choices=sorted(CASES), help="time ONE named workload and print its line")
    ap.add_argument("--sweep", action="store_true", help="configs[4] scaling sweep instead of the headline line")
    ap.add_argument("--sweep-max-log2", type=int, default=26)
    ap.add_argument("--plumbing-check", action="store_true", help="CPU-only: exercise the N-rank launch plumbing with gloo")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and not args.sweep and args.case is None:
        respawn_under_torchrun(args)
    if args.plumbing_check:
        run_plumbing_check(args)
    elif args.sweep:
        run_sweep(args)
    elif args.case is not None:
        run_case(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
