"""The tabulated anti-aliasing kernel handed to the gridder as an INPUT (plan argument).

BASELINE.json configs[0]: "prolate spheroidal (c = W*pi/2) tabulated in fp32 and normalised to unit
sum".  PAPER.md:27 (section 2.1) only says "a convolution that interpolates the samples onto a regular
grid"; the function, support and oversampling come from the configs (readings R5-R8).

psi_00(c, eta) is evaluated from its expansion in normalised even Legendre polynomials; the
coefficients are the eigenvector of the smallest eigenvalue of a symmetric tridiagonal matrix
(Flammer's recurrence written in the orthonormal basis sqrt(n+1/2) P_n).
"""
import numpy as np
from numpy.polynomial import legendre as _leg
from scipy.linalg import eigh_tridiagonal

_N_EVEN_TERMS = 60


def pswf_coefficients(c: float):
    """Return (chi0, beta): smallest eigenvalue and its eigenvector over n = 0, 2, 4, ..."""
    n = 2.0 * np.arange(_N_EVEN_TERMS)
    c2 = c * c
    diag = n * (n + 1.0) + c2 * (2.0 * n * (n + 1.0) - 1.0) / ((2.0 * n + 3.0) * (2.0 * n - 1.0))
    m = n[:-1]
    off = c2 * (m + 2.0) * (m + 1.0) / ((2.0 * m + 3.0) * np.sqrt((2.0 * m + 1.0) * (2.0 * m + 5.0)))
    w, v = eigh_tridiagonal(diag, off, select="i", select_range=(0, 0))
    beta = v[:, 0]
    if beta[0] < 0:
        beta = -beta
    return float(w[0]), beta


def pswf00(c: float, eta):
    """psi_00(c, eta) for |eta| <= 1 (arbitrary overall scale, positive at 0); 0 outside."""
    eta = np.asarray(eta, dtype=np.float64)
    _, beta = pswf_coefficients(c)
    coef = np.zeros(2 * _N_EVEN_TERMS)
    n = 2 * np.arange(_N_EVEN_TERMS)
    coef[n] = beta * np.sqrt(n + 0.5)
    inside = np.abs(eta) <= 1.0
    val = _leg.legval(np.where(inside, eta, 0.0), coef)
    return np.where(inside, val, 0.0)


def kernel_1d(W: int, x):
    """C(x) = psi_00(pi W / 2, 2x / W) for |x| <= W/2 cells, 0 outside (unscaled)."""
    x = np.asarray(x, dtype=np.float64)
    return pswf00(np.pi * W / 2.0, 2.0 * x / W)


def kernel_scale(W: int) -> float:
    """Global scale s that makes the centred row (offset 0) sum to 1."""
    h = (W - 1) // 2
    return 1.0 / float(np.sum(kernel_1d(W, np.arange(W) - h)))


def make_kernel_table(W: int, O: int) -> np.ndarray:
    """fp32 table T[ru][t], ru = 0..O, t = 0..W-1:  T[ru][t] = s * C((t - h) - (ru - O/2)/O).

    Row ru belongs to sub-cell offset r = ru - O/2 in [-O/2, O/2]; entry t is the kernel value at
    the distance from grid cell (ic + t - h) to the sample at ic + r/O.  The lower half is computed
    and the upper half mirrored so that T[O-ru][W-1-t] == T[ru][t] bit for bit.
    """
    if W % 2 != 1 or O % 2 != 0:
        raise ValueError("W must be odd and O even")
    h = (W - 1) // 2
    s = kernel_scale(W)
    T = np.zeros((O + 1, W), dtype=np.float32)
    t = np.arange(W, dtype=np.float64)
    for ru in range(O // 2 + 1):
        T[ru] = (s * kernel_1d(W, (t - h) - (ru - O // 2) / O)).astype(np.float32)
    T[O // 2] = 0.5 * (T[O // 2] + T[O // 2][::-1])          # exact mirror of the centred row
    for ru in range(O // 2 + 1, O + 1):
        T[ru] = T[O - ru][::-1]
    return np.ascontiguousarray(T)
