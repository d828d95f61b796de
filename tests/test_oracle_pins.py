"""Pins for the CPU oracle (DESIGN.md "Pins" P1, P3-P6 and the BASELINE.json fixed cases).

None of these compares the oracle with itself: expected values are worked by hand (golden file),
closed forms (a kernel stamp, flux sums, a direct DFT), symmetries, or an independently written
brute-force gather (oracle/brute.py shares no code with oracle/gridder.c).
"""
import numpy as np
import pytest

import oracle
from oracle import brute, imaging
from conftest import golden_rows
from gen import CONFIGS, generate, make_kernel_table, scaled

C = 299792458.0


def _grid(uv, freqs, vis, w, N, du, W, O, T):
    return oracle.grid(uv, freqs, vis, w, N, du, W, O, T, n_threads=2)


# ------------------------------------------------------------------ P1: the index formula
def test_p1_index_golden_table():
    for row in golden_rows("index_p1.txt"):
        x = float(row[0])
        for O, (wi, wr) in ((8, (int(row[1]), int(row[2]))), (16, (int(row[3]), int(row[4])))):
            i, r, ok = oracle.index(x, 256, 7, O)
            assert ok and (i, r) == (wi, wr), (x, O, i, r)
            i2, r2, ok2 = brute.index_np(np.array([x]), 256, 7, O)
            assert ok2[0] and (int(i2[0]), int(r2[0])) == (wi, wr)


def test_p1_edge_drop_and_nonfinite():
    # 124.5 -> i = 252, 252 + 3 = 255 <= 255 valid; 124.5625 -> i = 253, 256 > 255 dropped (R11)
    assert oracle.index(124.5, 256, 7, 8) == (252, 8, True)
    assert oracle.index(124.5625, 256, 7, 8) == (-1, -1, False)
    assert oracle.index(-124.5, 256, 7, 8) == (4, 0, True)          # 4 - 3 = 1 >= 0
    assert oracle.index(-125.5, 256, 7, 8) == (3, 0, True)          # ka = 1004 -> q = 125, rem = 4 stays inner
    assert oracle.index(-125.5625, 256, 7, 8)[2] is False           # ka = 1005 -> q = 126: i = 2, 2 - 3 < 0
    for bad in (np.nan, np.inf, -np.inf, 128.0, -128.0, 1e300):
        assert oracle.index(bad, 256, 7, 8) == (-1, -1, False)
    # W = 15: h = 7
    assert oracle.index(120.0, 256, 15, 16) == (248, 8, True)
    assert oracle.index(121.0, 256, 15, 16)[2] is False


@pytest.mark.parametrize("O", [2, 8, 16, 64])
def test_p1_index_properties(O):
    rs = np.random.RandomState(O)
    N, W = 4096, 7
    x = np.concatenate([rs.uniform(-2040, 2040, 20000), rs.randint(-2040 * O * 2, 2040 * O * 2, 20000) / (2.0 * O)])
    i, r, ok = brute.index_np(x, N, W, O)
    assert ok.all()
    ic, rr = i - N // 2, r - O // 2
    # quantised position within half a sub-cell, remainder range, exactly odd
    assert np.all(np.abs(x - (ic + rr / O)) <= 0.5 / O + 1e-12)
    assert rr.min() >= -O // 2 and rr.max() <= O // 2
    i2, r2, _ = brute.index_np(-x, N, W, O)
    assert np.array_equal(i2 - N // 2, -ic) and np.array_equal(r2 - O // 2, -rr)
    # the C function agrees with the numpy restatement value by value
    for k in range(0, x.size, 97):
        assert oracle.index(float(x[k]), N, W, O) == (int(i[k]), int(r[k]), True)


def test_indices_c_vs_numpy_on_c2_shape():
    g = generate(scaled(CONFIGS["C2"], n_ant=40, n_chan=5))
    cfg = g.cfg
    idx = oracle.compute_indices(g.uv, g.freqs, cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O)
    for c in range(cfg.n_chan):
        iu, iv, ru, rv, ok = brute.sample_indices(g.uv.numpy(), float(g.freqs[c]), cfg.grid_n, g.cell_du,
                                                  cfg.support_W, cfg.oversample_O)
        assert ok.all()
        assert np.array_equal(idx[:, c], np.stack([iu, iv, ru, rv], axis=1))


# ------------------------------------------------------------------ single visibility -> exact stamp
@pytest.mark.parametrize("W,O", [(7, 8), (15, 16)])
def test_single_visibility_reproduces_kernel_stamp(W, O):
    N, h = 256, (W - 1) // 2
    T = make_kernel_table(W, O)
    # s = 1 exactly, du = 1: x = u_m.  (10.0625, -10.25): O=8 -> (138,5),(118,2); O=16 -> (138,9),(118,4)
    uv = np.array([[10.0625, -10.25]])
    freqs = np.array([C])
    vis = np.array([[[1 + 0j, 2j, -3.0, 0.5 - 0.25j]]], dtype=np.complex64)
    G, A, _ = _grid(uv, freqs, vis, None, N, 1.0, W, O, T)
    ru, rv = (5, 2) if O == 8 else (9, 4)
    stamp = np.outer(T[rv].astype(np.float64), T[ru].astype(np.float64))      # [tv][tu]
    want = np.zeros((4, N, N), dtype=np.complex128)
    for p in range(4):
        want[p, 118 - h:118 + h + 1, 138 - h:138 + h + 1] = stamp * complex(vis[0, 0, p])
    assert np.array_equal(G[0], want)                                          # exact: one term per cell
    assert np.array_equal(A[0, 3], np.abs(want[3]))
    # weight scales everything, all pols alike
    G2, _, _ = _grid(uv, freqs, vis, np.array([[0.5]], dtype=np.float32), N, 1.0, W, O, T)
    assert np.array_equal(G2, 0.5 * G)


def test_dropped_sample_contributes_nothing_and_empty_input_zeroes():
    T = make_kernel_table(7, 8)
    uv = np.array([[124.5625, 0.0], [0.0, -126.0], [3.0, 4.0]])
    vis = np.ones((3, 1, 4), dtype=np.complex64)
    G, A, _ = _grid(uv, np.array([C]), vis, None, 256, 1.0, 7, 8, T)
    G1, _, _ = _grid(uv[2:], np.array([C]), vis[2:], None, 256, 1.0, 7, 8, T)
    assert np.array_equal(G, G1)
    idx = oracle.compute_indices(uv, np.array([C]), 256, 1.0, 7, 8)
    assert idx[0, 0].tolist() == [-1] * 4 and idx[1, 0].tolist() == [-1] * 4 and idx[2, 0].tolist() == [131, 132, 4, 4]
    G0, A0, _ = _grid(np.zeros((0, 2)), np.array([C]), np.zeros((0, 1, 4), np.complex64), None, 256, 1.0, 7, 8, T)
    assert not G0.any() and not A0.any()


# ------------------------------------------------------------------ P3 flux, linearity
@pytest.fixture(scope="module")
def c1():
    g = generate(CONFIGS["C1"])
    cfg = g.cfg
    G, A, _ = _grid(g.uv, g.freqs, g.vis, g.weights, cfg.grid_n, g.cell_du, cfg.support_W, cfg.oversample_O,
                    g.kernel_table)
    return g, G, A


def test_p3_flux_conservation(c1):
    g, G, A = c1
    cfg = g.cfg
    T = g.kernel_table.numpy().astype(np.float64)
    S = T.sum(axis=1)
    iu, iv, ru, rv, ok = brute.sample_indices(g.uv.numpy(), float(g.freqs[0]), cfg.grid_n, g.cell_du, 7, 8)
    assert ok.all()
    z = g.vis.numpy()[:, 0, :].astype(np.complex128) * g.weights.numpy()[:, 0:1].astype(np.float64)
    want = np.sum(z * (S[ru] * S[rv])[:, None], axis=0)
    got = G[0].sum(axis=(1, 2))
    assert np.all(np.abs(got - want) <= 1e-12 * np.abs(z).sum())
    wantA = np.sum(np.abs(z) * (S[ru] * S[rv])[:, None], axis=0)      # table entries are all >= 0
    assert np.allclose(A[0].sum(axis=(1, 2)), wantA, rtol=1e-12)


def test_linearity_in_v_and_w(c1):
    g, G, _ = c1
    cfg = g.cfg
    rs = np.random.RandomState(1)
    # inputs on a 2^-10 lattice so that 2*V1 - 0.5*V2 is exactly representable in complex64
    v1 = (np.round(g.vis.numpy() * 1024) / 1024).astype(np.complex64)
    v2 = ((rs.randint(-4096, 4096, g.vis.shape) + 1j * rs.randint(-4096, 4096, g.vis.shape)) / 1024).astype(np.complex64)
    args = (cfg.grid_n, g.cell_du, 7, 8, g.kernel_table)
    G1, _, _ = _grid(g.uv, g.freqs, v1, g.weights, *args)
    G2, _, _ = _grid(g.uv, g.freqs, v2, g.weights, *args)
    comb = (2.0 * v1.astype(np.complex128) - 0.5 * v2.astype(np.complex128))
    assert np.array_equal(comb.astype(np.complex64).astype(np.complex128), comb)
    G3, _, _ = _grid(g.uv, g.freqs, comb.astype(np.complex64), g.weights, *args)
    assert np.max(np.abs(G3 - (2.0 * G1 - 0.5 * G2))) <= 1e-13 * np.max(np.abs(G3))
    w2 = np.full(g.weights.shape, 0.25, dtype=np.float32)
    G4, _, _ = _grid(g.uv, g.freqs, g.vis, w2, *args)
    assert np.max(np.abs(G4 - 0.25 * G)) <= 1e-15 * np.max(np.abs(G))
    G5, _, _ = _grid(g.uv, g.freqs, g.vis, None, *args)              # NULL weights = ones (R12)
    assert np.array_equal(G5, G)


# ------------------------------------------------------------------ P4 Hermitian symmetry
def test_p4_conjugate_rows_give_hermitian_grid_and_real_image(c1):
    g, G, _ = c1
    N = g.cfg.grid_n
    body = G[0][:, 1:, 1:]                       # row/column 0 has no mirror partner on an even grid
    mirror = np.conj(body[:, ::-1, ::-1])
    assert np.max(np.abs(body - mirror)) <= 1e-15 * np.max(np.abs(G))
    assert not G[0][:, 0, :].any() and not G[0][:, :, 0].any()
    img = imaging.dirty_image(G[0])
    assert np.max(np.abs(img.imag)) <= 1e-13 * np.max(np.abs(img.real))


# ------------------------------------------------------------------ P6 brute-force gather
def test_p6_gather_equals_scatter_on_c1(c1):
    g, G, A = c1
    cfg = g.cfg
    Gg = brute.gather_grid(g.uv.numpy(), float(g.freqs[0]), g.vis.numpy()[:, 0], g.weights.numpy()[:, 0],
                           cfg.grid_n, g.cell_du, 7, 8, g.kernel_table.numpy())
    assert np.max(np.abs(Gg - G[0])) <= 1e-13 * np.max(np.abs(G))
    assert np.count_nonzero(G[0][0]) == np.count_nonzero(Gg[0]) > 1000


def test_p6_gather_cells_multichannel_w15():
    g = generate(scaled(CONFIGS["C5"], n_ant=16, core_ant=8, n_chan=3, grid_n=256))
    cfg = g.cfg
    G, A, _ = _grid(g.uv, g.freqs, g.vis, g.weights, cfg.grid_n, g.cell_du, 15, 16, g.kernel_table)
    rs = np.random.RandomState(5)
    nz = np.argwhere(A[2, 0] > 0)
    cells = [tuple(nz[k]) for k in rs.choice(len(nz), 60, replace=False)] + [(0, 0), (255, 255), (128, 128)]
    Gc, Ac = brute.gather_cells(g.uv.numpy(), float(g.freqs[2]), g.vis.numpy()[:, 2], g.weights.numpy()[:, 2],
                                cfg.grid_n, g.cell_du, 15, 16, g.kernel_table.numpy(), cells)
    for k, (j, i) in enumerate(cells):
        assert np.allclose(Gc[k], G[2, :, j, i], rtol=1e-12, atol=1e-13 * np.abs(G).max())
        assert np.allclose(Ac[k], A[2, :, j, i], rtol=1e-12)


# ------------------------------------------------------------------ P5 grid + FFT + correction vs direct DFT
@pytest.mark.parametrize("W,O,tol_q", [(7, 8, 2e-4), (15, 16, 1e-6)])
def test_p5_imaging_chain_matches_direct_dft(W, O, tol_q):
    g = generate(scaled(CONFIGS["C1"], support_W=W, oversample_O=O))
    cfg = g.cfg
    N = cfg.grid_n
    T = g.kernel_table.numpy()
    G, _, _ = _grid(g.uv, g.freqs, g.vis, g.weights, N, g.cell_du, W, O, T)
    ch = imaging.correction_1d(T, N, W, O)
    img = imaging.dirty_image(G[0, 0]).real / np.outer(ch, ch)
    uvn = g.uv.numpy()
    iu, iv, ru, rv, ok = brute.sample_indices(uvn, float(g.freqs[0]), N, g.cell_du, W, O)
    z = g.vis.numpy()[:, 0, 0].astype(np.complex128)
    s = float(g.freqs[0]) / C
    xq, yq = (iu - N // 2) + (ru - O // 2) / O, (iv - N // 2) + (rv - O // 2) / O
    xt, yt = uvn[:, 0] * s / g.cell_du, uvn[:, 1] * s / g.cell_du
    Dq = imaging.direct_dft(xq, yq, z, N).real
    Dt = imaging.direct_dft(xt, yt, z, N).real
    q = N // 4
    inner = slice(N // 2 - q, N // 2 + q)
    peak = np.abs(Dq).max()
    assert np.max(np.abs(img - Dq)[inner, inner]) <= tol_q * peak          # aliasing level of the kernel
    assert np.max(np.abs(img - Dt)[inner, inner]) <= 0.06 * np.abs(Dt).max()   # oversampling quantisation
    # sanity: the uncorrected image is far off, so the correction (and table addressing) matter
    raw = imaging.dirty_image(G[0, 0]).real
    assert np.max(np.abs(raw - Dq)[inner, inner]) > 0.05 * peak


# ------------------------------------------------------------------ f2: Stokes conversion
def test_stokes_oracle_against_the_textbook_definitions():
    from gen.stokes import S0, jones_field, mueller_of, stokes_matrix_field
    rs = np.random.RandomState(5)
    N, n_chan = 16, 3
    img = rs.standard_normal((n_chan, 4, N, N)) + 1j * rs.standard_normal((n_chan, 4, N, N))
    # (1) the constant textbook matrix: I = (XX + YY)/2, Q = (XX - YY)/2, U = (XY + YX)/2, V = -i (XY - YX)/2
    M0 = np.broadcast_to(S0, (N, N, 4, 4))
    s = imaging.stokes(img, M0)
    xx, xy, yx, yy = img[:, 0], img[:, 1], img[:, 2], img[:, 3]
    assert np.allclose(s[:, 0], (xx + yy) / 2) and np.allclose(s[:, 1], (xx - yy) / 2)
    assert np.allclose(s[:, 2], (xy + yx) / 2) and np.allclose(s[:, 3], -1j * (xy - yx) / 2)
    # (2) the identity leaves the planes alone; the map is linear; a transposed matrix (k <-> j) is caught
    eye = np.broadcast_to(np.eye(4), (N, N, 4, 4))
    assert np.array_equal(imaging.stokes(img, eye), img)
    assert np.allclose(imaging.stokes(2 * img + 1j * img[::-1], M0), 2 * s + 1j * imaging.stokes(img[::-1], M0))
    E = np.zeros((N, N, 4, 4)); E[..., 1, 2] = 1.0                  # out plane 1 <- in plane 2
    t = imaging.stokes(img, E)
    assert np.array_equal(t[:, 1], img[:, 2]) and not t[:, [0, 2, 3]].any()
    # (3) round trip through a direction-dependent instrument: known Stokes -> sky coherency -> J e J^H -> matrix field
    stokes_true = rs.standard_normal((n_chan, 4, N, N))
    coh = np.einsum("kj,cjqp->ckqp", np.linalg.inv(S0), stokes_true.astype(np.complex128))
    measured = np.einsum("qpkj,cjqp->ckqp", mueller_of(jones_field(N)), coh)
    back = imaging.stokes(measured, stokes_matrix_field(N).astype(np.complex128))
    assert np.allclose(back, stokes_true, atol=2e-6)               # the field is stored in complex64
    # per pixel: the matrix of pixel (q, p) is the one applied at (q, p)
    q, p = 3, 11
    M = stokes_matrix_field(N).astype(np.complex128)
    assert np.allclose(imaging.stokes(measured, M)[1, :, q, p], M[q, p] @ measured[1, :, q, p])


# ------------------------------------------------------------------ f3: general 2-D complex kernel tables
def _table_2d(T, phase=None):
    """[rv][ru][tv][tu] complex64 from the separable table T[(O+1)][W] (optionally times a per-tap phase screen)."""
    K = (T[:, None, :, None].astype(np.float64) * T[None, :, None, :].astype(np.float64)).astype(np.complex128)
    if phase is not None:
        K = K * np.exp(1j * phase)
    return K.astype(np.complex64)


def test_oracle_2d_tables_against_the_pinned_separable_gridder():
    N, W, O = 64, 7, 8
    T = make_kernel_table(W, O)
    rs = np.random.RandomState(8)
    n_vis, n_chan = 300, 2
    fr = np.array([299792458.0, 1.1 * 299792458.0])
    uv = rs.uniform(-24, 24, (n_vis, 2))
    vis = (rs.standard_normal((n_vis, n_chan, 4)) + 1j * rs.standard_normal((n_vis, n_chan, 4))).astype(np.complex64)
    wts = rs.uniform(0.5, 1.5, (n_vis, n_chan)).astype(np.float32)
    G1, A1, _ = oracle.grid(uv, fr, vis, wts, N, 1.0, W, O, T)
    # (1) a separable real table reproduces the 1-D gridder (up to the fp32 rounding of the stored products)
    G2, A2, _ = oracle.grid_2d(uv, fr, vis, wts, N, 1.0, W, O, _table_2d(T))
    assert np.all(np.abs(G2 - G1) <= 2e-7 * A1 + 1e-12) and np.allclose(A2, A1, rtol=2e-7)
    # (2) a constant phase factor on the kernel rotates the whole grid; (3) linearity in V
    G3, _, _ = oracle.grid_2d(uv, fr, vis, wts, N, 1.0, W, O, _table_2d(T, phase=0.7))
    assert np.all(np.abs(G3 - np.exp(0.7j) * G1) <= 4e-7 * A1 + 1e-12)
    G4, _, _ = oracle.grid_2d(uv, fr, (2 * vis).astype(np.complex64), wts, N, 1.0, W, O, _table_2d(T, phase=0.7))
    assert np.allclose(G4, 2 * G3, rtol=1e-12, atol=1e-14)
    # (4) one visibility stamps the [rv][ru] slice of a NON-separable complex table, tv along rows and tu along columns
    K = (rs.standard_normal((O + 1, O + 1, W, W)) + 1j * rs.standard_normal((O + 1, O + 1, W, W))).astype(np.complex64)
    uv1 = np.array([[10.0625, -10.25]])                              # pin P1: (iu, ru) = (42, 5), (iv, rv) = (22, 2) at N = 64
    v1 = np.zeros((1, 1, 4), dtype=np.complex64); v1[0, 0] = [1, 2j, -3, 0.5 - 0.25j]
    G5, A5, _ = oracle.grid_2d(uv1, fr[:1], v1, None, N, 1.0, W, O, K)
    h = 3
    for p in range(4):
        assert np.allclose(G5[0, p, 22 - h:22 + h + 1, 42 - h:42 + h + 1], K[2, 5].astype(np.complex128) * complex(v1[0, 0, p]), rtol=1e-15)
    assert np.count_nonzero(G5[0, 0]) == W * W and np.allclose(A5[0, 1, 22 - h:22 + h + 1, 42 - h:42 + h + 1], 2 * np.abs(K[2, 5]))
