"""Multi-GPU plumbing: the path shards trivially (every query / pixel is independent; PAPER.md:196 evaluates one
decoder query per pixel per light with no cross-query reduction), so ranks get disjoint batches, replicate the
~50 KB of weights and the latent table, and exchange NOTHING on the data path.  torch.distributed is used only for
the barrier around the timed region and the max-over-ranks of the device time."""
import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def rank_seed(base_seed, rank):
    """Weak scaling: rank r draws its own batch of the same shape from seed base_seed + 7919 * r."""
    return base_seed + 7919 * rank


def shard_range(n_items, rank, world):
    """Contiguous [lo, hi) slice of n_items for this rank (strong scaling of one batch / scanline blocks)."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_rows(height, rank, world, block=64):
    """Scanline block [row_lo, row_hi) of a frame for this rank: whole blocks of `block` rows (64 keeps the material tiles
    of the synthetic G-buffers whole), the blocks dealt out contiguously; the last rank takes the ragged remainder."""
    n_blocks = (height + block - 1) // block
    lo, hi = shard_range(n_blocks, rank, world)
    return min(height, lo * block), min(height, hi * block)


def all_gather_rows(local_rows, height, block=64):
    """Optional last step of a sharded frame: every rank ends up with the whole [height, width, C]
    image.  local_rows: this rank's [row_hi - row_lo, width, C] tensor (CPU tensor under gloo, CUDA tensor under nccl).
    Blocks are padded to the largest shard so that one all_gather serves ragged frames.  The only data-path collective in
    the package, and only for callers that need the assembled image on every GPU (24.9 MB at 1080p)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return local_rows
    world, rank = dist.get_world_size(), dist.get_rank()
    spans = [shard_rows(height, r, world, block) for r in range(world)]
    most = max(hi - lo for lo, hi in spans)
    pad = torch.zeros((most,) + tuple(local_rows.shape[1:]), dtype=local_rows.dtype, device=local_rows.device)
    pad[:local_rows.shape[0]] = local_rows
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][:hi - lo] for r, (lo, hi) in enumerate(spans)], dim=0)


def init(backend):
    import torch.distributed as dist
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """Max of a python float over all ranks (device time of the slowest rank)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device="cpu"):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
