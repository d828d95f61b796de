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


def abi_arguments(n_vis: int, n_chan: int, grid_n: int, world_size: int, rank: int) -> dict:
    """What `rank` hands to mwa_grid_visibilities when the call is sharded by channel (element offsets into the caller's
    full arrays; -> SURVEY.md section 8(e)): all uv rows, `n_chan` = its slice, its own planes of grid_out.
    vis / weights slices are strided in the [row][chan] layout, so the rank passes a contiguous copy of
    vis[:, c0:c1] / weights[:, c0:c1] (`vis_copy_elems` complex / `weights_copy_elems` floats)."""
    c0, c1 = channel_range(n_chan, world_size, rank)
    plane = grid_n * grid_n
    return {"rank": rank, "c0": c0, "c1": c1, "n_vis": n_vis, "n_chan": c1 - c0, "freqs_offset": c0,
            "vis_copy_elems": n_vis * (c1 - c0) * 4, "weights_copy_elems": n_vis * (c1 - c0),
            "grid_plane_offset": c0 * 4, "grid_planes": (c1 - c0) * 4,
            "grid_elem_offset": c0 * 4 * plane, "grid_elems": (c1 - c0) * 4 * plane}


def grid_channel_shard(plan, uv, freqs, vis, weights, world_size: int, rank: int, out=None, stream=None):
    """The channel-sharded driver (f4): grids this rank's channel slice with `plan` (a binding.Plan living on the rank's
    device) and returns (grids of the slice, (c0, c1)).  `out`, if given, is the FULL [n_chan, 4, N, N] grid on this
    device (single-node runs that keep one output array): the rank writes only its own planes of it.  No collective:
    ranks need no data from each other."""
    f, v, w, (c0, c1) = shard_inputs(freqs, vis, weights, world_size, rank)
    if c1 == c0:
        return (None if out is None else out[c0:c1]), (c0, c1)
    dev = uv.device
    f = f.to(dev).contiguous()
    v = v.to(dev).contiguous()
    w = None if w is None else w.to(dev).contiguous()
    target = None if out is None else out[c0:c1]                      # channel-major grid: a contiguous block of planes
    return plan.grid(uv, f, v, w, out=target, stream=stream), (c0, c1)
