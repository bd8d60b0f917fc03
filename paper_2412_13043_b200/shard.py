"""Sharding of a batch over ranks: every output of the library is independent, so a batch is
split along its external-point axis into contiguous blocks, one per rank, with no data-path collective.
`gather_blocks` is the optional epilogue when every rank wants the full result (an all-gather of the output
blocks: a few MiB over NVLink with NCCL, or gloo on CPU tensors)."""


def shard_bounds(n_units, world_size, rank):
    """[lo, hi) of rank's contiguous block; block sizes differ by at most one, earlier ranks get the larger ones."""
    if n_units < 0 or world_size < 1 or not (0 <= rank < world_size):
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_units, world_size)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def gather_blocks(local_block, n_units, dist):
    """All-gathers the per-rank blocks (axis 0 = external-point axis) into the full [n_units, ...] tensor.
    `dist` is torch.distributed (initialised); blocks may differ in length by one, so they are padded to the
    largest block for the collective and trimmed afterwards."""
    import torch
    world, rank = dist.get_world_size(), dist.get_rank()
    sizes = [shard_bounds(n_units, world, r) for r in range(world)]
    longest = max(hi - lo for lo, hi in sizes)
    lo, hi = sizes[rank]
    if local_block.shape[0] != hi - lo:
        raise ValueError("local block has %d rows, rank %d owns %d" % (local_block.shape[0], rank, hi - lo))
    pad = torch.zeros((longest,) + tuple(local_block.shape[1:]), dtype=local_block.dtype, device=local_block.device)
    pad[: hi - lo] = local_block
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][: sizes[r][1] - sizes[r][0]] for r in range(world)], dim=0)
