"""GPU parity: the CUDA library (through the C ABI binding) against the fp64 CPU oracle, same seeded inputs.

Indices must match bit for bit; grid values within the north_star tolerance (tests/parity.py).
Sizes: C1 and cut-down C2/C5 shapes element by element; C3 whole; C4 and C5 at FULL size on sampled
channels (a channel owns its grid, so a whole channel is compared element by element).
"""
import numpy as np
import pytest
import torch

import oracle
from gen import CONFIGS, generate, make_kernel_table, scaled
from parity import assert_parity

pytestmark = pytest.mark.gpu
C = 299792458.0
DESIGNS = ["atomic", "smem", "romein", "romein_sorted", "gather", "chan", "chanws"]


@pytest.fixture(scope="module")
def lib():
    from paper_0902_0915_b200 import _build
    _build.build()                      # no-op when the in-tree library is newer than its sources
    import paper_0902_0915_b200 as m
    return m


def _plan(lib, g, design="auto"):
    cfg = g.cfg
    return lib.Plan(cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O, g.kernel_table, design=design)


def _oracle(g, chans=None):
    cfg = g.cfg
    uv, fr, vis, w = g.uv.cpu(), g.freqs.cpu(), g.vis, g.weights
    if chans is not None:
        fr = fr[chans]
        vis = vis[:, chans]
        w = w[:, chans]
    return oracle.grid(uv, fr, vis.cpu(), w.cpu(), cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O,
                       g.kernel_table)


def _to_dev(g):
    g.uv, g.freqs, g.vis, g.weights = (t.cuda().contiguous() for t in (g.uv, g.freqs, g.vis, g.weights))
    return g


# ---------------------------------------------------------------------------- indices: bit-exact
@pytest.mark.parametrize("cfg", [CONFIGS["C1"], scaled(CONFIGS["C2"], n_ant=48, n_chan=7),
                                 scaled(CONFIGS["C5"], n_ant=24, core_ant=12, n_chan=5, grid_n=512),
                                 scaled(CONFIGS["C4"], n_ant=40, core_ant=20, n_chan=48, oversample_O=6)])
def test_indices_bit_exact(lib, cfg):
    g = generate(cfg)
    want = oracle.compute_indices(g.uv, g.freqs, cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O)
    _to_dev(g)
    with _plan(lib, g) as p:
        got = p.indices(g.uv, g.freqs).cpu().numpy()
    assert np.array_equal(got, want)


def test_indices_lattice_halfway_edges_and_nonfinite(lib):
    # positions on the 1/(2O) lattice hit every rounding tie; s = 1, du = 1 so x = u_m exactly
    N, W, O = 256, 7, 8
    lat = np.arange(-130 * 2 * O, 130 * 2 * O + 1) / (2.0 * O)
    rs = np.random.RandomState(3)
    extra = np.concatenate([rs.uniform(-130, 130, 5000), [np.nan, np.inf, -np.inf, 1e300, -0.0, 0.0, 124.5, 124.5625]])
    u = np.concatenate([lat, extra])
    uv = np.stack([u, u[::-1]], axis=1).copy()
    fr = np.array([C, 0.5 * C, 150e6])
    want = oracle.compute_indices(uv, fr, N, 1.0, W, O)
    with lib.Plan(N, 1.0, W, O, make_kernel_table(W, O)) as p:
        got = p.indices(torch.from_numpy(uv).cuda(), torch.from_numpy(fr).cuda()).cpu().numpy()
    assert np.array_equal(got, want)
    assert (want[:, 0, 0] == -1).any() and (want[:, 0, 0] >= 0).any()
    with lib.Plan(N, 1.0, W, O, make_kernel_table(W, O)) as p:                # the dropped-sample counter agrees with the oracle
        n_drop = lib.mwa_grid_count_dropped(p.handle, torch.from_numpy(uv).cuda(), torch.from_numpy(fr).cuda(), uv.shape[0], 3)
    assert n_drop == int((want[:, :, 0] == -1).sum()) and n_drop > 0


# ---------------------------------------------------------------------------- values
@pytest.mark.parametrize("design", DESIGNS)
def test_c1_whole_grid(lib, design):
    g = generate(CONFIGS["C1"])
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, design) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
        assert_parity(out.cpu().numpy(), G, A, design)
        out2 = p.grid(g.uv, g.freqs, g.vis, None)                 # NULL weights = ones (R12)
        assert_parity(out2.cpu().numpy(), G, A, design + " null weights")


@pytest.mark.parametrize("design", DESIGNS)
@pytest.mark.parametrize("name,kw", [
    ("C2", dict(n_ant=64, n_chan=6)),                              # several tiles, several channels
    ("C5", dict(n_ant=20, core_ant=10, n_chan=3, grid_n=512)),     # W = 15, O = 16, random weights, rotation
    ("C4", dict(n_ant=64, core_ant=32, n_chan=16, grid_n=250)),    # grid not a multiple of the tile: ragged tail
])
def test_cut_down_configs(lib, design, name, kw):
    if design == "chanws" and CONFIGS[name].support_W > 7:
        pytest.skip("K6's shared-memory budget holds the shifted table copies of W <= 7 kernels only (AUTO falls back to K5)")
    g = generate(scaled(CONFIGS[name], **kw))
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, design) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
    assert_parity(out.cpu().numpy(), G, A, f"{name} {design}")


@pytest.mark.parametrize("design", DESIGNS)
def test_c3_whole(lib, design):
    g = generate(CONFIGS["C3"], device="cuda")
    G, A, _ = _oracle(g)
    with _plan(lib, g, design) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
    assert_parity(out.cpu().numpy(), G, A, f"C3 {design}")


@pytest.mark.parametrize("design", ["chan", "chanws", "auto"])
@pytest.mark.parametrize("kw", [
    dict(n_ant=96, core_ant=48, n_chan=70, grid_n=512),            # 3 channel groups, the last one ragged (6 channels)
    dict(n_ant=200, core_ant=100, n_chan=33, grid_n=250),          # dense core -> multi-batch tiles; ragged grid edge
])
def test_fine_channels_c4_shape(lib, design, kw):
    # C4's 40 kHz channel spacing: the regime K5 (lane = channel) is built for, and the one AUTO must pick it in
    cfg = scaled(CONFIGS["C4"], **kw)
    cfg = scaled(cfg, f_lo_hz=155e6, f_hi_hz=155e6 + 40e3 * (cfg.n_chan - 1))
    g = generate(cfg)
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, design) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
        assert lib.mwa_grid_plan_last_design(p.handle) == ("chanws" if design == "auto" else design)
        assert_parity(out.cpu().numpy(), G, A, f"fine channels {design}")
        out2 = p.grid(g.uv, g.freqs, g.vis, None)
        assert_parity(out2.cpu().numpy(), G, A, f"fine channels {design} null weights")


def _fine(kw):
    cfg = scaled(CONFIGS["C4"], **kw)
    return scaled(cfg, f_lo_hz=155e6, f_hi_hz=155e6 + 40e3 * (cfg.n_chan - 1))


@pytest.mark.parametrize("design", ["chan", "chanws"])
@pytest.mark.parametrize("kw", [
    dict(n_ant=40, core_ant=20, n_chan=7 * 32 + 5, grid_n=128),    # K5: two super-groups, the second of 2 groups, last one ragged
    dict(n_ant=40, core_ant=20, n_chan=6 * 32 + 20, grid_n=128),   # K5: the second super-group is a single ragged group (dense path)
    dict(n_ant=24, core_ant=12, n_chan=1024 + 40, grid_n=64),      # more than 1024 channels: K5's group table moves to global memory
])
def test_many_channel_groups(lib, design, kw):
    # every group / super-group decode path of the channel-SIMD kernels, compared on ALL channels
    g = generate(_fine(kw))
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, design) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
        st = lib.mwa_grid_plan_last_stats(p.handle)
    assert st["error"] == 0
    assert_parity(out.cpu().numpy(), G, A, f"{design} {kw}")
    if design == "chan" and kw["n_chan"] == 6 * 32 + 20:
        assert st["k5_dense_items"] > 0                            # the single-group super-group took the dense path


def test_chanws_pool_overflow_takes_the_in_kernel_sweep(lib):
    # K6 sweeps an item itself when the pre-pass pool has no room for its hit list: same grid by a slower path
    g = generate(_fine(dict(n_ant=200, core_ant=100, n_chan=33, grid_n=250)))
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, "chanws") as p:
        ref = p.grid(g.uv, g.freqs, g.vis, g.weights).clone()
        st0 = lib.mwa_grid_plan_last_stats(p.handle)
        assert st0["swept_items"] == 0 and st0["max_hits"] > 64 and st0["error"] == 0
        for cap in (3000, 1):                                      # some items listed and some swept; (almost) all swept
            lib.mwa_grid_plan_set_list_pool(p.handle, cap)
            out = p.grid(g.uv, g.freqs, g.vis, g.weights)
            st = lib.mwa_grid_plan_last_stats(p.handle)
            assert st["swept_items"] > 0 and st["error"] == 0, st
            assert_parity(out.cpu().numpy(), G, A, f"pool capped at {cap}")
            assert st["items_with_hits"] == st0["items_with_hits"] and st["max_hits"] == st0["max_hits"]
        lib.mwa_grid_plan_set_list_pool(p.handle, 0)
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        assert torch.equal(out.view(torch.float32), ref.view(torch.float32))
        assert lib.mwa_grid_plan_last_stats(p.handle)["swept_items"] == 0


def test_auto_picks_gather_for_coarse_channels(lib):
    g = generate(scaled(CONFIGS["C2"], n_ant=32, n_chan=16, grid_n=256))     # 16 channels over 140-170 MHz
    _to_dev(g)
    with _plan(lib, g, "auto") as p:
        p.grid(g.uv, g.freqs, g.vis, g.weights)
        assert lib.mwa_grid_plan_last_design(p.handle) == "gather"


@pytest.mark.parametrize("design", ["chan", "chanws", "gather"])
def test_run_to_run_bit_identical(lib, design):
    # rows are put in a fixed order inside every uv bucket and neither product design uses atomics on grid data,
    # so two calls (and two plans) must agree bit for bit
    cfg = scaled(CONFIGS["C4"], n_ant=160, core_ant=80, n_chan=40, grid_n=512)
    cfg = scaled(cfg, f_lo_hz=155e6, f_hi_hz=155e6 + 40e3 * (cfg.n_chan - 1))
    g = _to_dev(generate(cfg))
    outs = []
    for _ in range(2):
        with _plan(lib, g, design) as p:
            outs.append(p.grid(g.uv, g.freqs, g.vis, g.weights).clone())
            outs.append(p.grid(g.uv, g.freqs, g.vis, g.weights).clone())
        torch.cuda.synchronize()
    for o in outs[1:]:
        assert torch.equal(outs[0].view(torch.float32), o.view(torch.float32))


def test_dense_tile_many_calls_on_one_plan(lib):
    # regression: the write-out stage of K5 aliases the visibility batch; without a barrier after the copy-out a
    # fast warp's cp.async for the next group could overwrite a slower warp's stage (seen once in ~10 calls)
    cfg = scaled(CONFIGS["C4"], n_ant=200, core_ant=100, n_chan=33, grid_n=250)
    cfg = scaled(cfg, f_lo_hz=155e6, f_hi_hz=155e6 + 40e3 * (cfg.n_chan - 1))
    g = generate(cfg)
    G, A, _ = _oracle(g)
    _to_dev(g)
    for design in ("auto", "chan"):
        with _plan(lib, g, design) as p:
            for k in range(12):
                out = p.grid(g.uv, g.freqs, g.vis, g.weights if k % 3 == 0 else None)
                assert_parity(out.cpu().numpy(), G, A, f"dense tile, {design}, call {k}")
            st = lib.mwa_grid_plan_last_stats(p.handle)
            assert st["error"] == 0
            if design == "chan":
                assert st["k5_dense_items"] > 0                    # K5 really took its dense-tile path
            else:
                assert st["max_hits"] > 6 * 16                     # K6: items longer than the whole staging ring


def test_chan_wide_kernel_repeated_calls(lib):
    # W = 15, O = 16 through K5; a second call on the same plan must pass parity too (workspace reuse)
    cfg = scaled(CONFIGS["C5"], n_ant=24, core_ant=12, n_chan=40, grid_n=512, f_lo_hz=150e6, f_hi_hz=150e6 + 39 * 40e3)
    g = generate(cfg)
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, "chan") as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        out2 = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
    assert_parity(out.cpu().numpy(), G, A, "chan W=15")
    assert_parity(out2.cpu().numpy(), G, A, "chan W=15, second call")


def test_c2_whole(lib):
    g = generate(CONFIGS["C2"], device="cuda")
    with _plan(lib, g) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
    for c0 in range(0, 32, 8):
        ch = list(range(c0, c0 + 8))
        G, A, _ = _oracle(g, ch)
        assert_parity(out[c0:c0 + 8].cpu().numpy(), G, A, f"C2 channels {c0}..")


def test_single_visibility_stamp_and_dropped_rows(lib):
    N, W, O, h = 256, 7, 8, 3
    T = make_kernel_table(W, O)
    uv = np.array([[10.0625, -10.25], [124.5625, 0.0], [0.0, -126.0], [-124.5, 124.5]])
    vis = np.zeros((4, 1, 4), dtype=np.complex64)
    vis[0, 0] = [1 + 0j, 2j, -3.0, 0.5 - 0.25j]
    vis[1:] = 7.0                                                  # rows 1, 2 are dropped whole (R11); row 3 is the last valid corner
    fr = np.array([C])
    G, A, _ = oracle.grid(uv, fr, vis, None, N, 1.0, W, O, T)
    for design in DESIGNS:
        with lib.Plan(N, 1.0, W, O, T, design=design) as p:
            out = p.grid(torch.from_numpy(uv).cuda(), torch.from_numpy(fr).cuda(), torch.from_numpy(vis).cuda())
            got = out.cpu().numpy()
        assert_parity(got, G, A, design)
        stamp = np.outer(T[2].astype(np.float64), T[5].astype(np.float64))    # rv = 2, ru = 5
        assert np.allclose(got[0, 0, 118 - h:118 + h + 1, 138 - h:138 + h + 1], stamp, rtol=3e-7, atol=0)
        assert np.count_nonzero(got[0, 0]) == 2 * W * W


@pytest.mark.parametrize("design", DESIGNS + ["auto"])
def test_dropped_samples_with_nonfinite_values_leave_no_trace(lib, design):
    # R11: a sample whose stamp leaves the grid is dropped whole - whatever its visibility and weight hold.  Flagged data
    # often carries NaN there; a kernel that multiplies it by a zero tap instead of skipping it would spread NaN.
    N, W, O = 256, 7, 8
    T = make_kernel_table(W, O)
    n_chan = 40
    fr = 155e6 + 40e3 * np.arange(n_chan)
    du = 1.0
    rs = np.random.RandomState(11)
    s0 = fr[0] / C
    edge = np.array([[124.4, 3.0], [-124.45, -60.2], [10.0, 124.3], [-124.0, 124.45], [123.9, -124.4]]) / s0   # valid at
    uv = np.concatenate([edge, rs.uniform(-100, 100, (300, 2)) / s0])      # channel 0, dropped further up the band
    idx = oracle.compute_indices(uv, fr, N, du, W, O)
    drop = idx[:, :, 0] < 0
    assert drop[:5].any() and not drop[:5].all() and not drop[5:].any()
    vis = (rs.standard_normal((uv.shape[0], n_chan, 4)) + 1j * rs.standard_normal((uv.shape[0], n_chan, 4))).astype(np.complex64)
    wts = rs.uniform(0.5, 1.5, (uv.shape[0], n_chan)).astype(np.float32)
    G, A, _ = oracle.grid(uv, fr, vis, wts, N, du, W, O, T)
    vis_bad, w_bad = vis.copy(), wts.copy()
    vis_bad[drop] = np.nan + 1j * np.inf
    w_bad[drop] = np.nan
    with lib.Plan(N, du, W, O, T, design=design) as p:
        t = [torch.from_numpy(x).cuda() for x in (uv, fr, vis_bad, w_bad)]
        out = p.grid(*t).cpu().numpy()
        assert np.isfinite(out.view(np.float32)).all(), design
        assert_parity(out, G, A, design)
        out2 = p.grid(t[0], t[1], t[2], None).cpu().numpy()              # NULL weights
        assert np.isfinite(out2.view(np.float32)).all(), design
    G1, A1, _ = oracle.grid(uv, fr, vis, None, N, du, W, O, T)
    assert_parity(out2, G1, A1, design + " null weights")


@pytest.mark.parametrize("design", ["gather", "chanws"])
def test_degenerate_input_with_a_huge_uv_bucket(lib, design):
    # 3000 rows inside one 8 x 8-cell uv bucket (plus a few elsewhere): above 2048 rows the in-bucket ordering switches from
    # ranking every row against every other one (quadratic: a million-row bucket would look like a hang) to a bitonic sort
    N, W, O = 128, 7, 8
    T = make_kernel_table(W, O)
    rs = np.random.RandomState(4)
    n_chan = 32 if design == "chanws" else 2
    fr = 155e6 + 40e3 * np.arange(n_chan)
    s0 = fr[-1] / C
    uv = np.concatenate([rs.uniform(16.5, 23.5, (3000, 2)), rs.uniform(-50, 50, (200, 2))]) / s0
    # partially coherent (random-sign terms would cancel and leave the Frobenius norm of the grid tiny; identical terms are
    # the worst case of sequential fp32 summation): unit amplitude, phases within +-1 rad; ~2300 terms per cell
    vis = np.exp(1j * rs.uniform(-1.0, 1.0, (uv.shape[0], n_chan, 4))).astype(np.complex64)
    G, A, _ = oracle.grid(uv, fr, vis, None, N, 1.0, W, O, T)
    with lib.Plan(N, 1.0, W, O, T, design=design) as p:
        t = [torch.from_numpy(x).cuda() for x in (uv, fr, vis)]
        out = p.grid(*t)
        out2 = p.grid(*t)
        assert torch.equal(out.view(torch.float32), out2.view(torch.float32))       # still a deterministic order
        assert_parity(out.cpu().numpy(), G, A, f"huge bucket {design}")


def test_empty_inputs_and_error_codes(lib):
    T = make_kernel_table(7, 8)
    with lib.Plan(64, 1.0, 7, 8, T) as p:
        fr = torch.tensor([C, 2 * C], dtype=torch.float64, device="cuda")
        out = torch.full((2, 4, 64, 64), 3 + 4j, dtype=torch.complex64, device="cuda")
        lib.mwa_grid_visibilities(p.handle, torch.zeros((0, 2), dtype=torch.float64, device="cuda"), fr,
                                  torch.zeros((0, 2, 4), dtype=torch.complex64, device="cuda"), None, 0, 2, out)
        assert not out.cpu().numpy().any()                          # n_vis == 0 zero-fills
        out.fill_(1)
        lib.mwa_grid_visibilities(p.handle, None, None, None, None, 0, 0, out)
        assert bool((out == 1).all())                               # n_chan == 0 is a no-op
        with pytest.raises(lib.MwaGridError) as e:
            lib.mwa_grid_visibilities(p.handle, torch.zeros((3, 2), dtype=torch.float64, device="cuda"), fr,
                                      None, None, 3, 2, out)
        assert e.value.code == -1 and "vis_c64" in str(e.value)
        with pytest.raises(lib.MwaGridError):
            lib.mwa_grid_visibilities(p.handle, None, fr, None, None, -1, 2, out)
    for bad in [(63, 1.0, 7, 8), (64, 0.0, 7, 8), (64, float("nan"), 7, 8), (64, 1.0, 6, 8), (64, 1.0, 7, 7),
                (64, 1.0, 17, 8), (8, 1.0, 7, 8)]:
        with pytest.raises(lib.MwaGridError):
            lib.mwa_grid_plan_create(bad[0], bad[1], bad[2], bad[3],
                                     np.zeros((bad[3] + 1) * bad[2], dtype=np.float32))


def test_host_entry_point_matches_device_call(lib):
    g = generate(scaled(CONFIGS["C2"], n_ant=32, n_chan=4, grid_n=256))
    G, A, _ = _oracle(g)
    cfg = g.cfg
    with _plan(lib, g) as p:
        out = torch.empty((cfg.n_chan, 4, cfg.grid_n, cfg.grid_n), dtype=torch.complex64).pin_memory()
        lib.mwa_grid_visibilities_host(p.handle, g.uv.pin_memory(), g.freqs.pin_memory(), g.vis.pin_memory(),
                                       g.weights.pin_memory(), cfg.n_vis, cfg.n_chan, out)
        assert_parity(out.numpy(), G, A, "host entry")
        assert lib.mwa_grid_plan_last_launches(p.handle) > 0


def test_host_entry_point_pipelined_over_channel_chunks(lib):
    # 100 fine channels -> 4 chunks (32, 32, 32, 4): upload, gridding and download of different chunks overlap
    g = generate(_fine(dict(n_ant=48, core_ant=24, n_chan=100, grid_n=128)))
    G, A, _ = _oracle(g)
    cfg = g.cfg
    with _plan(lib, g) as p:
        out = torch.full((cfg.n_chan, 4, cfg.grid_n, cfg.grid_n), float("nan"), dtype=torch.complex64).pin_memory()
        for weights in (g.weights.pin_memory(), None):
            out.fill_(float("nan"))
            lib.mwa_grid_visibilities_host(p.handle, g.uv.pin_memory(), g.freqs.pin_memory(), g.vis.pin_memory(), weights,
                                           cfg.n_vis, cfg.n_chan, out)
            assert_parity(out.numpy(), G, A, "host entry, 4 channel chunks")
        pageable = torch.empty_like(out)                                    # pageable buffers work too
        lib.mwa_grid_visibilities_host(p.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, pageable)
        assert_parity(pageable.numpy(), G, A, "host entry, pageable")


def test_plan_reuse_changing_sizes(lib):
    # workspace growth and reuse: small call, larger call, small again on the same plan
    T = make_kernel_table(7, 8)
    base = scaled(CONFIGS["C2"], n_ant=24, n_chan=2, grid_n=256)
    g_small, g_big = generate(base), generate(scaled(base, n_ant=72, n_chan=9))
    du = g_big.cell_du
    with lib.Plan(256, du, 7, 8, T) as p:
        for g in (g_small, g_big, g_small):
            G, A, _ = oracle.grid(g.uv, g.freqs, g.vis, g.weights, 256, du, 7, 8, T)
            out = p.grid(g.uv.cuda(), g.freqs.cuda(), g.vis.cuda(), g.weights.cuda())
            assert_parity(out.cpu().numpy(), G, A, "reuse")


# ---------------------------------------------------------------------------- full-size configs
def _indices_sampled(lib, p, g, chans):
    cfg = g.cfg
    idx = p.indices(g.uv, g.freqs[chans].contiguous()).cpu().numpy()
    want_idx = oracle.compute_indices(g.uv.cpu(), g.freqs[chans].cpu(), cfg.grid_n, g.cell_du, cfg.support_W,
                                      cfg.oversample_O)
    assert np.array_equal(idx, want_idx)


def test_c4_full_size_all_channels_and_run_to_run(lib):
    """The bench configuration, every one of the 768 channel grids compared with the oracle element by element (16
    channels at a time), every cell written, and the whole 25.8 GB grid bit-identical over repeated calls - with the
    deterministic hit order that is a whole-grid race detector."""
    g = generate(CONFIGS["C4"], device="cuda")
    cfg = g.cfg
    shape = (cfg.n_chan, 4, cfg.grid_n, cfg.grid_n)
    with _plan(lib, g) as p:
        out = torch.empty(shape, dtype=torch.complex64, device="cuda")
        out.fill_(float("nan"))
        lib.mwa_grid_visibilities(p.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, out)
        torch.cuda.synchronize()
        assert lib.mwa_grid_plan_last_design(p.handle) == "chanws"
        st = lib.mwa_grid_plan_last_stats(p.handle)
        assert st["error"] == 0 and st["swept_items"] == 0, st
        assert not bool(torch.isnan(out.view(torch.float32)).any())          # every cell of every plane was written
        _indices_sampled(lib, p, g, [0, 383, 767])
        again = torch.empty(shape, dtype=torch.complex64, device="cuda")
        for k in range(5):
            again.fill_(float("nan"))
            lib.mwa_grid_visibilities(p.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, again)
            assert torch.equal(out.view(torch.float32), again.view(torch.float32)), f"call {k} differs"
        del again
    worst = {"max_ratio": 0.0, "frob": 0.0}
    for c0 in range(0, cfg.n_chan, 16):
        ch = list(range(c0, min(c0 + 16, cfg.n_chan)))
        G, A, _ = _oracle(g, ch)
        r = assert_parity(out[c0:c0 + len(ch)].cpu().numpy(), G, A, f"C4 channels {c0}..{ch[-1]}")
        worst = {k: max(worst[k], r[k]) for k in worst}
    print("C4 full size, all channels:", worst)


def test_c5_full_size_sampled_channels(lib):
    g = generate(CONFIGS["C5"], device="cuda")
    cfg = g.cfg
    chans = [0, 31, 63]
    with _plan(lib, g) as p:
        out = torch.empty((cfg.n_chan, 4, cfg.grid_n, cfg.grid_n), dtype=torch.complex64, device="cuda")
        out.fill_(float("nan"))
        lib.mwa_grid_visibilities(p.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, out)
        torch.cuda.synchronize()
        _indices_sampled(lib, p, g, chans)
    assert not bool(torch.isnan(out.view(torch.float32)).any())              # every cell of every plane was written
    for c in chans:
        G, A, _ = _oracle(g, [c])
        assert_parity(out[c:c + 1].cpu().numpy(), G, A, f"C5 channel {c}")


# ---------------------------------------------------------------------------- f1: FFT + convolution correction
@pytest.mark.parametrize("W,O,tol_q", [(7, 8, 2e-4), (15, 16, 1e-6)])
@pytest.mark.parametrize("N", [256, 250])
def test_image_from_grid_matches_the_oracle_chain_and_the_direct_dft(lib, W, O, tol_q, N):
    """grid -> FFT -> correction on the GPU (mwa_image_from_grid) against (a) the same chain of the oracle, pixel by
    pixel, and (b) the brute-force DFT of the visibilities at SURVEY.md pin P5's levels (inner half of the image)."""
    from oracle import imaging
    cfg = scaled(CONFIGS["C1"], support_W=W, oversample_O=O, grid_n=N)
    g = generate(cfg)
    G, A, _ = _oracle(g)
    T = g.kernel_table
    ch = imaging.correction_1d(T.numpy(), N, W, O)
    want = imaging.dirty_image(G[0]) / np.outer(ch, ch)[None]                    # [4, N, N] complex128
    raw_peak = float(np.abs(imaging.dirty_image(G[0])).max())
    _to_dev(g)
    with _plan(lib, g) as p:
        got_ch = lib.mwa_image_correction(p.handle, N).numpy()
        assert np.allclose(got_ch, ch, rtol=1e-12, atol=1e-15)
        grid = p.grid(g.uv, g.freqs, g.vis, g.weights)
        img = p.image(grid)                                                       # out of place
        grid2 = grid.clone()
        p.image(grid2, out=grid2)                                                 # in place
        torch.cuda.synchronize()
        assert torch.equal(img.view(torch.float32), grid2.view(torch.float32))
    got = img[0].cpu().numpy().astype(np.complex128)
    # (a) fp32 gridding (<= 1e-5 A per cell) + fp32 FFT: a few 1e-6 of the raw peak, amplified by the correction
    bound = 2e-5 * raw_peak / np.abs(np.outer(ch, ch))[None]
    assert np.all(np.abs(got - want) <= bound), float(np.max(np.abs(got - want) / bound))
    # (b) pin P5 through the GPU: XX plane against the direct DFT at the quantised positions
    idx = oracle.compute_indices(g.uv.cpu(), g.freqs.cpu(), N, g.cell_du, W, O)[:, 0]
    ok = idx[:, 0] >= 0
    xq = (idx[ok, 0] - N // 2) + (idx[ok, 2] - O // 2) / O
    yq = (idx[ok, 1] - N // 2) + (idx[ok, 3] - O // 2) / O
    z = (g.weights.cpu().numpy()[ok, 0].astype(np.float64) * g.vis.cpu().numpy()[ok, 0, 0].astype(np.complex128))
    D = imaging.direct_dft(xq, yq, z, N)
    lo, hi = N // 2 - N // 4, N // 2 + N // 4
    err = np.abs(got[0, lo:hi, lo:hi] - D[lo:hi, lo:hi]).max() / np.abs(D).max()
    # W = 7: the kernel's aliasing level (2e-4).  W = 15: the fp64 oracle chain reaches 1e-6 (tests/test_oracle_pins.py); the
    # GPU chain is fp32 (gridding 1e-5 A per cell, cuFFT single precision) and the correction amplifies its rounding by
    # up to 1 / c^(N/4)^2 = 450 at the corner of the inner half: measured 1.9e-6, bound 5e-6
    assert err <= max(tol_q, 5e-6), err


# ---------------------------------------------------------------------------- f4: channel-sharded driver
def test_channel_sharded_driver_matches_the_unsharded_call(lib):
    """Two (and three) ranks' calls, run one after the other on this one GPU, write disjoint planes of one grid_out that
    passes parity against the oracle's whole-band grid.  (Not bit-identical to the unsharded call: a call bins its rows at
    its OWN top frequency, so a shard sums the same taps in another order.)"""
    from paper_0902_0915_b200.shard import grid_channel_shard
    g = generate(_fine(dict(n_ant=64, core_ant=32, n_chan=100, grid_n=256)))
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g) as p:
        for ws in (2, 3):
            out = torch.full((g.cfg.n_chan, 4, g.cfg.grid_n, g.cfg.grid_n), float("nan"), dtype=torch.complex64, device="cuda")
            covered = []
            for rank in range(ws):
                part, (c0, c1) = grid_channel_shard(p, g.uv, g.freqs, g.vis, g.weights, ws, rank, out=out)
                assert part.data_ptr() == out[c0:c1].data_ptr()
                covered += list(range(c0, c1))
            torch.cuda.synchronize()
            assert covered == list(range(g.cfg.n_chan))
            assert_parity(out.cpu().numpy(), G, A, f"{ws} channel shards")


# ---------------------------------------------------------------------------- f2: Stokes conversion
@pytest.mark.parametrize("N,n_chan", [(64, 5), (250, 2)])
def test_stokes_conversion_matches_the_oracle(lib, N, n_chan):
    from gen.stokes import stokes_matrix_field
    from oracle import imaging
    rs = np.random.RandomState(9)
    img = (rs.standard_normal((n_chan, 4, N, N)) + 1j * rs.standard_normal((n_chan, 4, N, N))).astype(np.complex64)
    M = stokes_matrix_field(N)
    want = imaging.stokes(img, M)
    bound = 1e-6 * np.einsum("qpkj,cjqp->ckqp", np.abs(M).astype(np.float64), np.abs(img).astype(np.float64)) + 1e-9
    with lib.Plan(N, 1.0, 7, 8, make_kernel_table(7, 8)) as p:
        d_img, d_M = torch.from_numpy(img).cuda(), torch.from_numpy(M).cuda()
        out = p.stokes(d_img, d_M)
        assert np.all(np.abs(out.cpu().numpy().astype(np.complex128) - want) <= bound)      # 16 fp32 FMAs per output
        inplace = d_img.clone()
        p.stokes(inplace, d_M, out=inplace)
        assert torch.equal(inplace.view(torch.float32), out.view(torch.float32))


# ---------------------------------------------------------------------------- f3: accumulate-into
@pytest.mark.parametrize("design", ["auto", "gather", "chanws", "atomic", "romein"])
@pytest.mark.parametrize("fine", [True, False])
def test_accumulate_into_adds_row_batches_onto_one_grid(lib, design, fine):
    """Two row batches gridded one after the other with accumulate-into equal the oracle's grid of all rows (the
    aggregation in time of PAPER.md:23), and what the grid held before is kept, not overwritten."""
    if fine:
        g = generate(_fine(dict(n_ant=64, core_ant=32, n_chan=40, grid_n=250)))
    else:
        if design == "chanws":
            pytest.skip("coarse channels: covered by the other designs")
        g = generate(scaled(CONFIGS["C2"], n_ant=48, n_chan=5, grid_n=256))
    G, A, _ = _oracle(g)
    _to_dev(g)
    half = g.cfg.n_vis // 2
    rs = np.random.RandomState(2)
    prev = (rs.standard_normal(G.shape) + 1j * rs.standard_normal(G.shape)).astype(np.complex64)
    with _plan(lib, g, design) as p:
        lib.mwa_grid_plan_set_accumulate(p.handle, True)
        out = torch.from_numpy(prev).cuda()
        for r0, r1 in ((0, half), (half, g.cfg.n_vis)):
            p.grid(g.uv[r0:r1].contiguous(), g.freqs, g.vis[r0:r1].contiguous(), g.weights[r0:r1].contiguous(), out=out)
        got = out.cpu().numpy()
        lib.mwa_grid_plan_set_accumulate(p.handle, False)
        again = p.grid(g.uv, g.freqs, g.vis, g.weights, out=out).cpu().numpy()    # back to overwrite (R10)
    want = prev.astype(np.complex128) + G
    # the fp32 tolerance of the gridded part, plus one rounding of the running sum per call
    bound = 1e-5 * A + 1e-7 + 3 * 2.0 ** -24 * (np.abs(prev) + np.abs(want))
    assert np.all(np.abs(got.astype(np.complex128) - want) <= bound), float(np.max(np.abs(got - want) / bound))
    assert_parity(again, G, A, f"{design} overwrite after accumulate")


# ---------------------------------------------------------------------------- f3: multi-frequency synthesis
@pytest.mark.parametrize("design", ["auto", "gather", "atomic", "romein", "romein_sorted"])
def test_multi_frequency_synthesis_sums_the_channels_onto_one_grid(lib, design):
    g = generate(scaled(CONFIGS["C2"], n_ant=48, n_chan=12, grid_n=250))
    G, A, _ = _oracle(g)
    G, A = G.sum(axis=0, keepdims=True), A.sum(axis=0, keepdims=True)      # the definition: one grid = sum over channels
    _to_dev(g)
    with _plan(lib, g, design) as p:
        p.set_mfs(True)
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        assert tuple(out.shape) == (1, 4, 250, 250)
        assert_parity(out.cpu().numpy(), G, A, f"MFS {design}")
        lib.mwa_grid_plan_set_accumulate(p.handle, True)                    # MFS + accumulate-into: a second pass doubles it
        p.grid(g.uv, g.freqs, g.vis, g.weights, out=out)
        assert_parity(out.cpu().numpy(), 2 * G, 2 * A, f"MFS {design} accumulated twice")
        lib.mwa_grid_plan_set_accumulate(p.handle, False)
        p.set_mfs(False)
        back = p.grid(g.uv, g.freqs, g.vis, g.weights)                      # and back to one grid per channel
        assert tuple(back.shape) == (12, 4, 250, 250)


def test_grid_out_aligned_to_16_but_not_32_bytes(lib):
    """The ABI asks for a 16-byte aligned grid_out; K3c's 256-bit stores need 32 and must fall back to 128-bit stores."""
    g = generate(scaled(CONFIGS["C2"], n_ant=48, n_chan=3, grid_n=256))
    cfg = g.cfg
    G, A, _ = _oracle(g)
    _to_dev(g)
    n = cfg.n_chan * 4 * cfg.grid_n * cfg.grid_n
    buf = torch.full((n + 2,), complex(float("nan"), float("nan")), dtype=torch.complex64, device="cuda")
    out = buf[2:].view(cfg.n_chan, 4, cfg.grid_n, cfg.grid_n)              # 16 bytes past a 512-byte aligned allocation
    assert out.data_ptr() % 32 == 16
    with _plan(lib, g, "gather") as p:
        lib.mwa_grid_visibilities(p.handle, g.uv, g.freqs, g.vis, g.weights, cfg.n_vis, cfg.n_chan, out)
        torch.cuda.synchronize()
        assert_parity(out.cpu().numpy(), G, A, "gather, grid_out 16-byte aligned")
        ref = p.grid(g.uv, g.freqs, g.vis, g.weights)                         # 32-byte aligned: the 256-bit path
        assert torch.equal(ref.view(torch.float32), out.contiguous().view(torch.float32))
    assert torch.isnan(buf[:2].real).all()                                   # nothing written in front of the grid


# ---------------------------------------------------------------------------- K3c: heavy tiles gridded by four warps
@pytest.mark.parametrize("mode", ["overwrite", "accumulate", "mfs"])
def test_gather_heavy_tiles_are_gridded_by_the_four_warps_of_a_cta(lib, mode):
    """Few items per warp and a dense core (C3's regime): K3c takes the items of the heavy tiles first, one per CTA, every warp
    a quarter of the candidates, partial tiles added in a fixed order.  Observable through last_stats; bit-identical from
    call to call; all three write-out modes."""
    g = generate(scaled(CONFIGS["C3"], n_ant=128, core_ant=96, core_radius_m=300.0, n_chan=2, grid_n=500,
                        f_lo_hz=150e6, f_hi_hz=152e6))             # 22 tiles of 256 - 1900 rows each
    assert g.cfg.n_vis > 4096                                        # not the one-CTA pre-pass of small calls
    G, A, _ = _oracle(g)
    _to_dev(g)
    with _plan(lib, g, "gather") as p:
        if mode == "mfs":
            p.set_mfs(True)
            G, A = G.sum(axis=0, keepdims=True), A.sum(axis=0, keepdims=True)
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
        st = lib.mwa_grid_plan_last_stats(p.handle)
        assert st["k3c_heavy_items"] > 0, st
        assert_parity(out.cpu().numpy(), G, A, f"heavy tiles {mode}")
        for _ in range(3):
            again = p.grid(g.uv, g.freqs, g.vis, g.weights)
            if mode != "mfs":                                        # MFS adds the channels with reductions: order not fixed
                assert torch.equal(again.view(torch.float32), out.view(torch.float32))
        if mode == "accumulate":
            lib.mwa_grid_plan_set_accumulate(p.handle, True)
            p.grid(g.uv, g.freqs, g.vis, g.weights, out=out)
            bound = 2 * (1e-5 * A + 1e-7) + 3 * 2.0 ** -24 * np.abs(2 * G)
            assert np.all(np.abs(out.cpu().numpy().astype(np.complex128) - 2 * G) <= bound)
            lib.mwa_grid_plan_set_accumulate(p.handle, False)


# ---------------------------------------------------------------------------- K6 stress: many shapes, repeated calls
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_chanws_random_shapes_repeated_calls(lib, seed):
    """compute-sanitizer is not available on the GPU pool, so races in K6's mbarrier pipeline are hunted by repetition: random
    grid sizes (ragged edges), antenna counts (sparse to dense tiles) and channel counts (ragged last group, many
    groups), each gridded three times on one plan - bit-identical every time and within tolerance of the oracle."""
    rs = np.random.RandomState(100 + seed)
    for _ in range(4):
        n_ant = int(rs.choice([12, 40, 90, 180]))
        kw = dict(n_ant=n_ant, core_ant=n_ant // 2, n_chan=int(rs.choice([8, 31, 32, 45, 96, 130])),
                  grid_n=int(rs.choice([64, 96, 250, 256, 384])))
        g = generate(_fine(kw))
        G, A, _ = _oracle(g)
        _to_dev(g)
        with _plan(lib, g, "chanws") as p:
            first = p.grid(g.uv, g.freqs, g.vis, g.weights).clone()
            for k in range(2):
                again = p.grid(g.uv, g.freqs, g.vis, g.weights)
                assert torch.equal(first.view(torch.float32), again.view(torch.float32)), (kw, k)
            assert lib.mwa_grid_plan_last_stats(p.handle)["error"] == 0
        assert_parity(first.cpu().numpy(), G, A, f"K6 stress {kw}")


# ---------------------------------------------------------------------------- f3: companion weights grid
def test_weights_grid_equals_the_grid_of_unit_visibilities(lib):
    g = generate(scaled(CONFIGS["C5"], n_ant=24, core_ant=12, n_chan=3, grid_n=250))        # random weights, W = 15
    ones = np.ones((g.cfg.n_vis, g.cfg.n_chan, 4), dtype=np.complex64)
    G, A, _ = oracle.grid(g.uv, g.freqs, ones, g.weights, g.cfg.grid_n, g.cell_du, g.cfg.support_W, g.cfg.oversample_O,
                          g.kernel_table)
    _to_dev(g)
    with _plan(lib, g) as p:
        wg = torch.full((g.cfg.n_chan, 250, 250), float("nan"), dtype=torch.float32, device="cuda")
        lib.mwa_grid_weights_grid(p.handle, g.uv, g.freqs, g.weights, g.cfg.n_vis, g.cfg.n_chan, wg)
        got = wg.cpu().numpy().astype(np.float64)
        wg1 = torch.empty_like(wg)
        lib.mwa_grid_weights_grid(p.handle, g.uv, g.freqs, None, g.cfg.n_vis, g.cfg.n_chan, wg1)   # NULL weights = ones
    want, bound = G[:, 0].real, 1e-5 * A[:, 0] + 1e-7                    # the XX plane of the unit-visibility grid
    assert np.all(np.abs(got - want) <= bound), float(np.max(np.abs(got - want) / bound))
    assert np.count_nonzero(got[A[:, 0] == 0]) == 0
    G1, A1, _ = oracle.grid(g.uv.cpu(), g.freqs.cpu(), ones, None, g.cfg.grid_n, g.cell_du, g.cfg.support_W, g.cfg.oversample_O,
                            g.kernel_table)
    assert np.all(np.abs(wg1.cpu().numpy() - G1[:, 0].real) <= 1e-5 * A1[:, 0] + 1e-7)


# ---------------------------------------------------------------------------- f3: general 2-D complex kernel tables
@pytest.mark.parametrize("name,kw", [
    ("C2", dict(n_ant=48, n_chan=5, grid_n=250)),                          # W = 7, O = 8, ragged grid edge
    ("C5", dict(n_ant=20, core_ant=10, n_chan=2, grid_n=256)),             # W = 15, O = 16, random weights
])
def test_2d_complex_kernel_table(lib, name, kw):
    g = generate(scaled(CONFIGS[name], **kw))
    cfg = g.cfg
    W, O = cfg.support_W, cfg.oversample_O
    rs = np.random.RandomState(13)
    T = g.kernel_table.numpy().astype(np.float64)
    # a non-separable complex kernel: the separable one times a tap- and row-dependent phase screen, plus a small random part
    K = T[:, None, :, None] * T[None, :, None, :] * np.exp(1j * rs.uniform(-1.5, 1.5, (O + 1, O + 1, W, W)))
    K = (K + 0.01 * (rs.standard_normal(K.shape) + 1j * rs.standard_normal(K.shape)) * np.abs(K).max()).astype(np.complex64)
    G, A, _ = oracle.grid_2d(g.uv, g.freqs, g.vis, g.weights, cfg.grid_n, g.cell_du, W, O, K)
    _to_dev(g)
    with lib.Plan(cfg.grid_n, g.cell_du, W, O, K, table_2d=True) as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        again = p.grid(g.uv, g.freqs, g.vis, g.weights)
        assert torch.equal(out.view(torch.float32), again.view(torch.float32))
        assert_parity(out.cpu().numpy(), G, A, f"2-D table {name}")
        idx = p.indices(g.uv, g.freqs).cpu().numpy()                        # the same index function
        with pytest.raises(lib.MwaGridError):
            p.image(out)
    assert np.array_equal(idx, oracle.compute_indices(g.uv.cpu(), g.freqs.cpu(), cfg.grid_n, g.cell_du, W, O))
