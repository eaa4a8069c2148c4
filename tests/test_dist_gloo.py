"""world_size-2 gloo test of the N>1 plumbing (CPU): disjoint per-rank batches, contiguous shard ranges that
tile the whole batch, max-over-ranks timing, and per-rank oracle results that concatenate to the whole-batch result."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import oracle
    from paper_2406_17782_b200 import dist, synth
    r, _, w = dist.init("gloo")
    assert (r, w) == (rank, world)
    cfg = synth.config(1, n=1001)
    lo, hi = dist.shard_range(1001, r, w)
    part = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"][lo:hi], n_threads=1)
    dist.barrier()
    t = dist.max_over_ranks(10.0 + rank)
    total = dist.sum_over_ranks(hi - lo)
    seed = dist.rank_seed(1, r)
    own = synth.config(1, n=64, seed=seed)["queries"]
    q.put((rank, lo, hi, part, t, total, own["u"][:4].copy()))
    dist.finalize()


def _frame_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import oracle
    from paper_2406_17782_b200 import dist, synth
    dist.init("gloo")
    cfg = synth.config(2, width=48, height=150)              # 150 rows: blocks of 64, 64, 22 -> a ragged last shard
    g, W = cfg["gbuffer"], 48
    lo, hi = dist.shard_rows(150, rank, world)
    part = oracle.shade_frame(cfg["weights"], cfg["biases"], cfg["latents"], g, cfg["lights"], first=lo * W,
                              count=(hi - lo) * W, n_threads=1)
    whole = dist.all_gather_rows(torch.from_numpy(part.reshape(hi - lo, W, 3)), 150)
    q.put((rank, lo, hi, whole.numpy()))
    dist.finalize()


def test_two_rank_scanline_blocks_and_frame_all_gather():
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_frame_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=180) for _ in procs], key=lambda x: x[0])
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2406_17782_b200 import synth
    cfg = synth.config(2, width=48, height=150)
    ref = oracle.shade_frame(cfg["weights"], cfg["biases"], cfg["latents"], cfg["gbuffer"], cfg["lights"]).reshape(150, 48, 3)
    assert (res[0][1], res[0][2], res[1][1], res[1][2]) == (0, 128, 128, 150)        # whole 64-row blocks, ragged tail last
    for r in res:
        np.testing.assert_array_equal(r[3], ref)                                      # every rank holds the whole image


def test_two_rank_sharding_and_timing_reduction():
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in procs], key=lambda x: x[0])
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    sys.path.insert(0, ROOT)
    import oracle
    from paper_2406_17782_b200 import synth
    cfg = synth.config(1, n=1001)
    whole = oracle.eval_queries(cfg["weights"], cfg["biases"], cfg["latents"], cfg["queries"])
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == 1001          # ranges tile the batch
    np.testing.assert_array_equal(np.concatenate([res[0][3], res[1][3]]), whole)    # no cross-query coupling
    assert res[0][4] == res[1][4] == 11.0 and res[0][5] == res[1][5] == 1001.0
    assert not np.array_equal(res[0][6], res[1][6])                                  # weak scaling: distinct batches
