"""Shared helpers of the GPU parity tests: the tolerance of BASELINE.json north_star, written out.

  per cell   |gpu - oracle| <= 1e-5 * A + 1e-7,  A = sum |w| |c| |V| of the taps landing in the cell
  per call   ||gpu - oracle||_F / ||oracle||_F <= 1e-6

The oracle side (G in complex128, A in float64) comes from oracle/gridder.c only.
"""
import numpy as np

REL_CELL = 1e-5
ABS_CELL = 1e-7
REL_FROB = 1e-6


def compare(G_gpu, G_ref, A_ref):
    """Returns a dict of error measures; G_gpu complex64 array, G_ref complex128, A_ref float64 (same shape)."""
    G_gpu = np.asarray(G_gpu)
    diff = np.abs(G_gpu.astype(np.complex128) - G_ref)
    bound = REL_CELL * A_ref + ABS_CELL
    ratio = float(np.max(diff / bound)) if diff.size else 0.0
    nrm = float(np.linalg.norm(G_ref.ravel()))
    frob = float(np.linalg.norm((G_gpu.astype(np.complex128) - G_ref).ravel()) / nrm) if nrm > 0 else 0.0
    untouched = A_ref == 0
    return {"max_ratio": ratio, "frob": frob, "max_abs": float(diff.max()) if diff.size else 0.0,
            "nonzero_where_untouched": int(np.count_nonzero(G_gpu[untouched]))}


def assert_parity(G_gpu, G_ref, A_ref, what=""):
    r = compare(G_gpu, G_ref, A_ref)
    assert r["nonzero_where_untouched"] == 0, (what, r)         # cells no tap reaches must be exact zeros (R10)
    assert r["max_ratio"] <= 1.0, (what, r)
    assert r["frob"] <= REL_FROB, (what, r)
    return r
