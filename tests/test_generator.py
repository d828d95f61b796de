"""Generator checks: the kernel table (pin P2) and the shape/statistics of the synthetic inputs."""
import numpy as np
import pytest
from scipy.special import pro_ang1

from conftest import golden_rows
from gen import CONFIGS, generate, scaled
from gen.pswf import kernel_scale, make_kernel_table, pswf00, pswf_coefficients
from gen import rng
import torch


@pytest.mark.parametrize("W", [7, 15])
def test_pswf_matches_scipy_and_golden(W):
    c = np.pi * W / 2
    eta = np.linspace(0.0, 0.999, 41)
    ours = pswf00(c, eta) / pswf00(c, 0.0)
    ref = np.array([pro_ang1(0, 0, c, e)[0] for e in eta]) / pro_ang1(0, 0, c, 0.0)[0]
    assert np.max(np.abs(ours - ref)) < 1e-9
    for row in golden_rows("pswf_p2.txt"):
        if row[0] == "chi":
            if int(row[1]) == W:
                assert abs(pswf_coefficients(c)[0] - float(row[2])) < 1e-9
        elif int(row[0]) == W:
            e, want = float(row[1]), float(row[2])
            got = float(pswf00(c, e) / pswf00(c, 0.0))
            assert abs(got - want) <= 2e-6 * want + 1e-15, (W, e, got, want)


@pytest.mark.parametrize("W,O", [(7, 8), (15, 16)])
def test_kernel_table_structure(W, O):
    T = make_kernel_table(W, O)
    assert T.shape == (O + 1, W) and T.dtype == np.float32
    # R8: mirror symmetry bit for bit
    assert np.array_equal(T[::-1, ::-1], T)
    # R7: centred row sums to one; others within the aliasing level
    assert abs(T[O // 2].sum(dtype=np.float64) - 1.0) < 2e-7
    assert np.all(np.abs(T.sum(axis=1, dtype=np.float64) - 1.0) < (2e-4 if W == 7 else 2e-7))
    # end rows are the same samples shifted by one tap
    assert np.allclose(T[0][:-1], T[O][1:], rtol=0, atol=1e-7)
    # table entry = s*C(distance)
    h = (W - 1) // 2
    s = kernel_scale(W)
    c = np.pi * W / 2
    for ru in (0, 1, O // 2, O - 1):
        d = (np.arange(W) - h) - (ru - O // 2) / O
        want = s * pswf00(c, 2 * d / W)
        assert np.allclose(T[ru], want, rtol=0, atol=1e-7)


def test_kernel_table_golden_values():
    # SURVEY.md section 8(c) P2 "fp32 table rows"
    T = make_kernel_table(7, 8)
    assert np.allclose(T[4][:4], [0.0029764287, 0.061112754, 0.24692975, 0.37796214], rtol=2e-7)
    assert np.allclose(T[0], [1.8216103e-2, 1.4136142e-1, 3.4033915e-1, 3.4033915e-1, 1.4136142e-1,
                              1.8216103e-2, 7.2731636e-5], rtol=3e-7)
    assert abs(T.sum(dtype=np.float64) - 8.99983298) < 1e-6
    T = make_kernel_table(15, 16)
    assert np.allclose(T[8][7:], [0.25819889, 0.21063964, 0.11311627, 0.038564391, 0.0077540539,
                                  7.9582189e-4, 3.0232412e-5, 1.4619036e-7], rtol=3e-7)
    assert abs(T.sum(dtype=np.float64) - 17.00000003) < 1e-6


def test_rng_is_counter_based_and_uniform():
    idx = torch.arange(200000)
    u = rng.uniform(7, 3, idx)
    assert torch.equal(u[1000:2000], rng.uniform(7, 3, idx[1000:2000]))       # chunk-independent
    assert 0.0 < float(u.min()) and float(u.max()) < 1.0
    assert abs(float(u.mean()) - 0.5) < 5e-3 and abs(float(u.var()) - 1 / 12) < 2e-3
    g = rng.normal(7, 3, idx)
    assert abs(float(g.mean())) < 1e-2 and abs(float(g.std()) - 1.0) < 1e-2
    assert not torch.equal(u, rng.uniform(8, 3, idx))


def test_config_shapes_match_baseline():
    want = {"C1": (992, 3968, 194432), "C2": (16256, 2080768, 101957632), "C3": (261632, 1046528, 51279872),
            "C4": (130816, 401866752, 19691470848), "C5": (1046528, 267911168, 60280012800)}
    for k, (nv, vp, taps) in want.items():
        c = CONFIGS[k]
        assert (c.n_vis, c.vis_pol(), c.tap_updates()) == (nv, vp, taps)
    assert abs(CONFIGS["C4"].algorithmic_bytes() / 1e9 - 29.389) < 1e-3
    f = CONFIGS["C4"].freqs()
    assert abs(float(f[1] - f[0]) - 40e3) < 1e-3 and abs(float(f.mean()) - 155e6) < 1.0


def test_generate_c1_properties():
    g = generate(CONFIGS["C1"])
    cfg = g.cfg
    assert g.uv.shape == (992, 2) and g.vis.shape == (992, 1, 4) and g.vis.dtype == torch.complex64
    # conjugate rows: (-u,-v), conj(V)
    assert torch.equal(g.uv[496:], -g.uv[:496]) and torch.equal(g.vis[496:], g.vis[:496].conj())
    # 90 % rule: nothing is dropped and the largest coordinate sits at 0.45 N cells
    x = g.uv * (float(g.freqs.max()) / 299792458.0) / g.cell_du
    assert abs(float(x.abs().max()) - 0.45 * cfg.grid_n) < 1e-9
    # deterministic
    g2 = generate(CONFIGS["C1"])
    assert torch.equal(g.vis, g2.vis) and torch.equal(g.uv, g2.uv)
    # chunking does not change the result beyond fp64 summation order
    g3 = generate(CONFIGS["C1"], rows_per_chunk=37)
    assert torch.allclose(g.vis, g3.vis, rtol=0, atol=1e-6)


def test_generate_rotation_and_weights_small_c5():
    cfg = scaled(CONFIGS["C5"], n_ant=12, core_ant=6, n_chan=3, grid_n=256)
    g = generate(cfg)
    nb = cfg.n_baselines
    assert g.uv.shape == (8 * nb, 2)
    # consecutive integrations move a baseline only slightly (8 s of earth rotation)
    step = (g.uv[nb:2 * nb] - g.uv[:nb]).norm(dim=1) / g.uv[:nb].norm(dim=1)
    assert float(step.max()) < 1e-3 and float(step.max()) > 0
    assert 0.5 <= float(g.weights.min()) and float(g.weights.max()) <= 1.5
    assert abs(float(g.weights.mean()) - 1.0) < 0.1
