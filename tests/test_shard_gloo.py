"""N > 1 host logic on CPU: two gloo ranks partition the channels (no data-path collective), each would grid its own
slice; the only exchanges are the bench's barrier and the max-over-ranks of the step time."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_0902_0915_b200.shard import GROUP, abi_arguments, channel_range, shard_inputs


def test_channel_ranges_cover_every_channel_once():
    for n_chan in [0, 1, 31, 32, 33, 70, 768, 1000]:
        for ws in [1, 2, 3, 8, 32]:
            got = []
            for r in range(ws):
                c0, c1 = channel_range(n_chan, ws, r)
                assert 0 <= c0 <= c1 <= n_chan
                assert c0 % GROUP == 0 or c0 == n_chan
                got += list(range(c0, c1))
            assert got == list(range(n_chan)), (n_chan, ws)
    sizes = [channel_range(768, 32, r) for r in range(32)]
    assert all(c1 - c0 == 24 or (c1 - c0) % GROUP == 0 for c0, c1 in sizes)      # 32 nodes


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, ws, port, n_vis, n_chan, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    g = torch.Generator().manual_seed(7)                              # every rank builds the same synthetic input
    freqs = torch.linspace(140e6, 170e6, n_chan, dtype=torch.float64)
    vis = torch.randn((n_vis, n_chan, 4), dtype=torch.complex64, generator=g)
    wts = torch.rand((n_vis, n_chan), generator=g)
    f, v, w, (c0, c1) = shard_inputs(freqs, vis, wts, ws, rank)
    assert f.shape[0] == c1 - c0 and v.shape[1] == c1 - c0 and w.shape[1] == c1 - c0
    # what the bench exchanges: a barrier and the max over ranks of the step time; the per-rank channel sums stand in
    # for "each rank wrote its own grid planes" and must add up to the whole without any overlap
    dist.barrier()
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    part = torch.zeros(n_chan, dtype=torch.complex128)
    part[c0:c1] = (v.to(torch.complex128) * w[..., None]).sum(dim=(0, 2))
    parts = [torch.zeros_like(part) for _ in range(ws)]
    dist.all_gather(parts, part)                                      # test-only exchange
    # the argument list each rank would hand to the C ABI (f4): rank 0 checks that the plane ranges tile grid_out
    grid_n = 64
    a = abi_arguments(n_vis, n_chan, grid_n, ws, rank)
    assert a["n_chan"] == c1 - c0 and a["freqs_offset"] == c0 and a["vis_copy_elems"] == v.numel()
    assert a["weights_copy_elems"] == w.numel() and a["grid_elem_offset"] % (grid_n * grid_n) == 0
    mine = torch.tensor([a["grid_elem_offset"], a["grid_elems"], a["grid_plane_offset"], a["grid_planes"]], dtype=torch.int64)
    every = [torch.zeros_like(mine) for _ in range(ws)]
    dist.all_gather(every, mine)
    if rank == 0:
        pos = 0
        for e in every:                                               # ranks in order: contiguous, no gap, no overlap
            assert int(e[0]) == pos and int(e[2]) * grid_n * grid_n == pos
            pos += int(e[1])
        assert pos == n_chan * 4 * grid_n * grid_n
    if rank == 0:
        whole = (vis.to(torch.complex128) * wts[..., None]).sum(dim=(0, 2))
        out.put((float(t.item()), bool(torch.allclose(sum(parts), whole)),
                 int(sum((p != 0).sum() for p in parts))))
    dist.destroy_process_group()


def test_two_gloo_ranks_shard_channels_without_overlap():
    ws, n_vis, n_chan = 2, 50, 70
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, ws, port, n_vis, n_chan, out)) for r in range(ws)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    tmax, ok, nonzero = res
    assert tmax == 2.0 and ok and nonzero == n_chan                   # max over ranks; planes add up; no overlap
