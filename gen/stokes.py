"""Synthetic per-pixel 4x4 matrix field for the Stokes-conversion step.

The paper says the matrix "is a function of time and position on the sky relative to the instrument and must be calculated
... for each pixel" and gives no formula, so the library takes it as an input (R18) and this module only makes a
smooth, well-conditioned stand-in: M(l, m) = S0 . inverse(J (x) conj(J)) with the textbook coherency -> Stokes matrix S0
and an analytic direction-dependent Jones matrix J(l, m).  An input generator: it holds none of the library's arithmetic.
"""
import numpy as np

# (I, Q, U, V) from the coherency vector (XX, XY, YX, YY) of linear feeds
S0 = 0.5 * np.array([[1, 0, 0, 1], [1, 0, 0, -1], [0, 1, 1, 0], [0, -1j, 1j, 0]], dtype=np.complex128)


def jones_field(N: int, fov: float = 0.6):
    """[N, N, 2, 2] complex128: J(l, m) on the image pixel grid, l, m in [-fov/2, fov/2)."""
    ax = (np.arange(N) - N // 2) * (fov / N)
    m, l = np.meshgrid(ax, ax, indexing="ij")                      # row q <-> m, column p <-> l
    J = np.empty((N, N, 2, 2), dtype=np.complex128)
    J[..., 0, 0] = 1.0 - 0.5 * l * l + 0.05j * m
    J[..., 0, 1] = 0.3 * l * m + 0.02j * l
    J[..., 1, 0] = -0.25 * l * m + 0.03j * m
    J[..., 1, 1] = 1.0 - 0.5 * m * m - 0.04j * l
    return J


def mueller_of(J):
    """[..., 4, 4]: J (x) conj(J), the matrix that takes the sky coherency vector to the measured one."""
    return np.einsum("...ab,...cd->...acbd", J, np.conj(J)).reshape(J.shape[:-2] + (4, 4))


def stokes_matrix_field(N: int, fov: float = 0.6):
    """[N, N, 4, 4] complex64: measured (XX, XY, YX, YY) -> (I, Q, U, V) for every pixel."""
    K = mueller_of(jones_field(N, fov))
    return (S0[None, None] @ np.linalg.inv(K)).astype(np.complex64)
