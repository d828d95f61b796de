"""TEST INFRASTRUCTURE - brute-force "gather" restatement of the gridding sum in numpy (fp64).

PAPER.md:49 describes the gather form: "a thread collects the values for a particular memory
location".  Here one grid cell collects, from ALL samples, the taps that land on it.  Written
independently of gridder.c (no shared code) so that the two pin each other (DESIGN.md pin P6),
and cheap enough per cell to check sampled cells of the full-size configs.
"""
import numpy as np

C_LIGHT = 299792458.0


def index_np(x, N, W, O):
    """Vectorised INDEX(x) (R4): returns (i, r, ok) arrays; i, r are -1 where dropped."""
    x = np.asarray(x, dtype=np.float64)
    h = (W - 1) // 2
    inside = np.abs(x) < N // 2                      # False for NaN
    a = np.where(inside, np.abs(x), 0.0)
    sgn = np.where(np.signbit(x), -1, 1).astype(np.int64)
    ka = np.floor(a * float(O) + 0.5).astype(np.int64)
    q, rem = ka // O, ka % O
    up = rem > O // 2
    q = np.where(up, q + 1, q)
    rem = np.where(up, rem - O, rem)
    i = N // 2 + sgn * q
    r = sgn * rem + O // 2
    ok = inside & (i - h >= 0) & (i + h <= N - 1)
    return np.where(ok, i, -1), np.where(ok, r, -1), ok


def sample_indices(uv, freq_hz, N, du, W, O):
    """(iu, iv, ru, rv, ok) of every row at one frequency; x = (u_m * (nu/c)) * (1/du)  (R3)."""
    uv = np.asarray(uv, dtype=np.float64)
    s = np.float64(freq_hz) / np.float64(C_LIGHT)
    inv_du = np.float64(1.0) / np.float64(du)
    iu, ru, oku = index_np((uv[:, 0] * s) * inv_du, N, W, O)
    iv, rv, okv = index_np((uv[:, 1] * s) * inv_du, N, W, O)
    ok = oku & okv
    return iu, iv, ru, rv, ok


def gather_cells(uv, freq_hz, vis_c, weights_c, N, du, W, O, table, cells):
    """Value and |.|-sum of chosen cells of ONE channel.

    vis_c [n_vis,4] complex, weights_c [n_vis] or None, cells = iterable of (j, i) = (row v, col u).
    Returns (G [len(cells),4] complex128, A [len(cells),4] float64)."""
    h = (W - 1) // 2
    T = np.asarray(table, dtype=np.float64)
    iu, iv, ru, rv, ok = sample_indices(uv, freq_hz, N, du, W, O)
    z = np.asarray(vis_c, dtype=np.complex128)
    if weights_c is not None:
        z = z * np.asarray(weights_c, dtype=np.float64)[:, None]
    cells = list(cells)
    G = np.zeros((len(cells), 4), dtype=np.complex128)
    A = np.zeros((len(cells), 4), dtype=np.float64)
    for k, (j, i) in enumerate(cells):
        tv, tu = j - iv + h, i - iu + h
        hit = ok & (tv >= 0) & (tv < W) & (tu >= 0) & (tu < W)
        n = np.nonzero(hit)[0]
        if n.size == 0:
            continue
        kern = T[rv[n], tv[n]] * T[ru[n], tu[n]]
        G[k] = np.sum(kern[:, None] * z[n], axis=0)
        A[k] = np.sum(np.abs(kern)[:, None] * np.abs(z[n]), axis=0)
    return G, A


def gather_grid(uv, freq_hz, vis_c, weights_c, N, du, W, O, table):
    """Whole plane set of one channel by per-cell gathering (tiny inputs only): [4,N,N] complex128."""
    cells = [(j, i) for j in range(N) for i in range(N)]
    G, _ = gather_cells(uv, freq_hz, vis_c, weights_c, N, du, W, O, table, cells)
    return G.reshape(N, N, 4).transpose(2, 0, 1).copy()
