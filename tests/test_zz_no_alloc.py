"""mwa_grid_visibilities_noalloc - the gridding call that allocates nothing (static device scratch, csrc/k_noalloc.cu) -
against the existing plan path (design GATHER, the same kernels on a cudaMalloc'ed workspace).

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide other tests).  Self-contained:
passes alone in a fresh process and after the other test files.
"""
import numpy as np
import pytest
import torch

import oracle
from gen import CONFIGS, generate, scaled
from parity import ABS_CELL, REL_CELL, REL_FROB

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lib():
    from paper_0902_0915_b200 import _build
    _build.build()                      # no-op when the in-tree library is newer than its sources
    import paper_0902_0915_b200 as m
    return m


def _case(cfg):
    g = generate(cfg)
    _, A, _ = oracle.grid(g.uv.cpu(), g.freqs.cpu(), g.vis.cpu(), g.weights.cpu(), cfg.grid_n, g.cell_du, cfg.support_W,
                          cfg.oversample_O, g.kernel_table)          # A = sum |w||c||V| per cell: the tolerance's scale
    g.uv, g.freqs, g.vis, g.weights = (t.cuda().contiguous() for t in (g.uv, g.freqs, g.vis, g.weights))
    g.table_dev = torch.as_tensor(np.asarray(g.kernel_table), dtype=torch.float32).cuda().contiguous()
    return g, A


def _plan_path(lib, g):
    cfg = g.cfg
    with lib.Plan(cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O, g.kernel_table, design="gather") as p:
        out = p.grid(g.uv, g.freqs, g.vis, g.weights)
        torch.cuda.synchronize()
        return out.clone()


def _noalloc(lib, g, out):
    cfg = g.cfg
    lib.mwa_grid_visibilities_noalloc(cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O, g.table_dev, g.uv, g.freqs,
                                      g.vis, g.weights, cfg.n_vis, cfg.n_chan, out)


def _assert_close(got, ref, A, what):
    got, ref = got.cpu().numpy().astype(np.complex128), ref.cpu().numpy().astype(np.complex128)
    assert np.all(np.isfinite(got.view(np.float64))), what             # the NaN pre-fill is gone: every cell was written
    # the parity tolerance of tests/parity.py (north_star): per cell 1e-5 * A + 1e-7, per call 1e-6 in Frobenius norm
    assert np.max(np.abs(got - ref) / (REL_CELL * A + ABS_CELL)) <= 1.0, what
    assert np.linalg.norm((got - ref).ravel()) <= REL_FROB * np.linalg.norm(ref.ravel()), what
    assert np.count_nonzero(got[A == 0]) == 0, what


def test_noalloc_entry_point_matches_the_plan_path_on_two_calls_in_a_row(lib):
    # a: ragged grid, 5310 rows x 5 channels, W = 15 (multi-kernel binning path); b: C1 (single-CTA binning path), smaller in
    # every dimension, so the second call runs on the stale scratch contents of the first
    ga, Aa = _case(scaled(CONFIGS["C5"], n_ant=60, core_ant=30, n_int=3, n_chan=5, grid_n=250))
    gb, Ab = _case(CONFIGS["C1"])
    ref_a, ref_b = _plan_path(lib, ga), _plan_path(lib, gb)
    nan = float("nan")
    out_a = torch.full_like(ref_a, complex(nan, nan))
    out_b = torch.full_like(ref_b, complex(nan, nan))
    out_a2 = torch.full_like(ref_a, complex(nan, nan))
    _noalloc(lib, ga, torch.empty_like(ref_a))           # set-up call: resolves the symbol, loads the kernels
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    _noalloc(lib, ga, out_a)                             # two calls in a row on one stream, then the first again
    _noalloc(lib, gb, out_b)
    _noalloc(lib, ga, out_a2)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before                     # nothing was allocated on the device by the three calls
    _assert_close(out_a, ref_a, Aa, "first call")
    _assert_close(out_b, ref_b, Ab, "second call")
    _assert_close(out_a2, ref_a, Aa, "third call")
    # the same kernels in the same order: bit for bit the plan's GATHER design
    assert torch.equal(out_a.view(torch.float32), ref_a.view(torch.float32))
    assert torch.equal(out_b.view(torch.float32), ref_b.view(torch.float32))
    assert torch.equal(out_a2.view(torch.float32), out_a.view(torch.float32))


def test_noalloc_entry_point_rejects_sizes_beyond_the_static_scratch(lib):
    g, _ = _case(CONFIGS["C1"])
    cfg = g.cfg
    out = torch.zeros(cfg.n_chan, 4, cfg.grid_n, cfg.grid_n, dtype=torch.complex64, device="cuda")
    before = out.clone()

    def call(grid_n=cfg.grid_n, n_vis=cfg.n_vis, n_chan=cfg.n_chan):
        lib.mwa_grid_visibilities_noalloc(grid_n, g.cell_du, cfg.support_W, cfg.oversample_O, g.table_dev, g.uv, g.freqs,
                                          g.vis, g.weights, n_vis, n_chan, out)

    for kw, name in (({"n_vis": lib.NOALLOC_MAX_VIS + 1}, "MWA_GRID_NOALLOC_MAX_VIS"),
                     ({"n_chan": lib.NOALLOC_MAX_CHAN + 1}, "MWA_GRID_NOALLOC_MAX_CHAN"),
                     ({"grid_n": lib.NOALLOC_MAX_GRID_N + 2}, "MWA_GRID_NOALLOC_MAX_GRID_N")):
        with pytest.raises(lib.MwaGridError) as e:
            call(**kw)
        assert name in str(e.value) and e.value.code == -1, str(e.value)     # MWA_GRID_ERR_INVALID, nothing enqueued
    torch.cuda.synchronize()
    assert torch.equal(out.view(torch.float32), before.view(torch.float32))
    call(n_vis=0)                                        # n_vis == 0 zero-fills; n_chan == 0 is a no-op
    call(n_chan=0)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0
