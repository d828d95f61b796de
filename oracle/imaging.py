"""TEST INFRASTRUCTURE - the steps after gridding, used only to pin the gridder (DESIGN.md pin P5).

PAPER.md:27 says the grid exists "to permit the operation of the Fast Fourier Transform"; Table 1
 lists FFT and "Convolution Correction" as the next two tasks.  A gridder with a wrong
sign, centre or table addressing does not survive grid -> FFT -> correction -> compare with a direct DFT.
"""
import numpy as np


def dirty_image(G):
    """I[q][p] = sum_{j,i} G[j][i] exp(+2 pi i ((i-N/2) p + (j-N/2) q)/N), p,q in [-N/2, N/2)."""
    N = G.shape[-1]
    return np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(G, axes=(-2, -1))), axes=(-2, -1)) * (N * N)


def correction_1d(table, N, W, O):
    """c^(p) = (1/O) sum_k C(k/O) cos(2 pi (k/O) p / N), k = -WO/2..WO/2, end terms halved.

    The samples C(k/O) are read back from the table itself: T[ru][t] = C((t-h) - (ru-O/2)/O)."""
    T = np.asarray(table, dtype=np.float64)
    h = (W - 1) // 2
    half = W * O // 2
    k = np.arange(-half, half + 1)
    vals = np.empty(k.size)
    for n, kk in enumerate(k):
        m = int(min(max(np.floor(kk / O + 0.5), -h), h))     # tap t - h, an integer in [-h, h]
        r = m * O - int(kk)                                  # sub-cell offset in [-O/2, O/2]
        vals[n] = T[r + O // 2, m + h]
    wts = np.ones(k.size)
    wts[0] = wts[-1] = 0.5
    p = np.arange(-N // 2, N // 2)
    return (1.0 / O) * np.sum(wts[None] * vals[None] * np.cos(2 * np.pi * np.outer(p, k / O) / N), axis=1)


def direct_dft(x_cells, y_cells, z, N):
    """D[q][p] = sum_n z_n exp(+2 pi i (x_n p + y_n q)/N), x,y in cells relative to the grid centre."""
    p = np.arange(-N // 2, N // 2)
    ex = np.exp(2j * np.pi * np.outer(x_cells, p) / N)      # [n, p]
    ey = np.exp(2j * np.pi * np.outer(y_cells, p) / N)      # [n, q]
    return np.einsum("n,nq,np->qp", np.asarray(z, dtype=np.complex128), ey, ex)


def stokes(image, matrix):
    """"converted into a set of Stokes parameters by the application of a 4x4 matrix transformation ...
    calculated ... for each pixel".  out[c][k][q][p] = sum_j matrix[q][p][k][j] * image[c][j][q][p], in complex128."""
    return np.einsum("qpkj,cjqp->ckqp", np.asarray(matrix, dtype=np.complex128), np.asarray(image, dtype=np.complex128))
