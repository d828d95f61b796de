"""Channel sharding for more than one GPU (PAPER.md:37 plans 32 GPU nodes for 768 channels).

Every channel owns its grids, so the path shards by channel with NO collective: a rank needs all uv rows, its
slice of `freqs`, the channel slice of `vis` / `weights`, and writes only its own `grid_out` planes.  The partition is
contiguous and aligned to 32 channels (the lane = channel kernel works on groups of 32 adjacent channels), with the
remainder spread over the first ranks.  Host logic only - no arithmetic of the method lives here.
"""
GROUP = 32


def channel_range(n_chan: int, world_size: int, rank: int):
    """[c0, c1) of `rank`: contiguous, GROUP-aligned starts, sizes differ by at most one group."""
    if world_size < 1 or not (0 <= rank < world_size) or n_chan < 0:
        raise ValueError("bad world_size / rank / n_chan")
    n_groups = (n_chan + GROUP - 1) // GROUP
    base, extra = divmod(n_groups, world_size)
    g0 = rank * base + min(rank, extra)
    g1 = g0 + base + (1 if rank < extra else 0)
    return min(g0 * GROUP, n_chan), min(g1 * GROUP, n_chan)


def shard_inputs(freqs, vis, weights, world_size: int, rank: int):
    """Views of one rank's channel slice: (freqs[c0:c1], vis[:, c0:c1], weights[:, c0:c1] or None, (c0, c1)).
    The slices of vis / weights are strided in the [row][chan] layout; call .contiguous() before the ABI."""
    c0, c1 = channel_range(int(freqs.shape[0]), world_size, rank)
    w = None if weights is None else weights[:, c0:c1]
    return freqs[c0:c1], vis[:, c0:c1], w, (c0, c1)
