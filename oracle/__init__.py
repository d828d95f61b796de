"""TEST INFRASTRUCTURE - CPU oracle for convolutional visibility gridding (section 2.1).

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this package.  It shares no code with `paper_0902_0915_b200` and never imports it.

  gridder.c   the definition as fp64 scatter loops (the authority; built here with gcc)
  brute.py    per-cell "gather" restatement in numpy for tiny inputs / sampled cells
  imaging.py  dirty image, grid correction and direct DFT used by pin P5

Parity of the oracle against the paper's own (unpublished) gridder output: UNPINNED.
Pinned against the mathematics by tests/test_oracle_*.py - see DESIGN.md "Pins".
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gridder.c")
_LIB = os.path.join(_HERE, "liboracle_gridder.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile gridder.c with gcc (no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P = ctypes.c_void_p
        lib.oracle_index.argtypes = [ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
        lib.oracle_index.restype = ctypes.c_int
        lib.oracle_compute_indices.argtypes = [P, P, ctypes.c_longlong, ctypes.c_int, ctypes.c_int,
                                               ctypes.c_double, ctypes.c_int, ctypes.c_int, P]
        lib.oracle_compute_indices.restype = None
        lib.oracle_grid.argtypes = [P, P, P, P, ctypes.c_longlong, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_double, ctypes.c_int, ctypes.c_int, P, P, P, ctypes.c_int]
        lib.oracle_grid.restype = ctypes.c_int
        lib.oracle_grid_2d.argtypes = lib.oracle_grid.argtypes
        lib.oracle_grid_2d.restype = ctypes.c_int
        _lib = lib
    return _lib


def _np(x, dtype):
    if hasattr(x, "detach"):
        x = x.detach().cpu().numpy()
    return np.ascontiguousarray(x, dtype=dtype)


def index(x: float, grid_n: int, support_W: int, oversample_O: int):
    """INDEX(x) -> (i, r, ok) for one coordinate already expressed in cells."""
    i, r = ctypes.c_int(), ctypes.c_int()
    ok = _load().oracle_index(float(x), grid_n, support_W, oversample_O, ctypes.byref(i), ctypes.byref(r))
    return i.value, r.value, bool(ok)


def compute_indices(uv, freqs, grid_n, cell_du, support_W, oversample_O) -> np.ndarray:
    """[n_vis, n_chan, 4] int32 = (iu, iv, ru, rv), or -1s for a dropped sample."""
    uv, freqs = _np(uv, np.float64), _np(freqs, np.float64)
    n_vis, n_chan = uv.shape[0], freqs.shape[0]
    out = np.empty((n_vis, n_chan, 4), dtype=np.int32)
    _load().oracle_compute_indices(uv.ctypes.data, freqs.ctypes.data, n_vis, n_chan, grid_n,
                                   float(cell_du), support_W, oversample_O, out.ctypes.data)
    return out


def grid(uv, freqs, vis, weights, grid_n, cell_du, support_W, oversample_O, kernel_table,
         want_abs: bool = True, n_threads: int = 0):
    """Grid all channels.  Returns (G complex128 [n_chan,4,N,N], A float64 [n_chan,4,N,N] or None, threads)."""
    uv, freqs = _np(uv, np.float64), _np(freqs, np.float64)
    vis = _np(vis, np.complex64)
    n_vis, n_chan = uv.shape[0], freqs.shape[0]
    assert vis.shape == (n_vis, n_chan, 4), vis.shape
    w_ptr = None
    if weights is not None:
        weights = _np(weights, np.float32)
        assert weights.shape == (n_vis, n_chan)
        w_ptr = weights.ctypes.data
    table = _np(kernel_table, np.float32)
    assert table.shape == (oversample_O + 1, support_W)
    G = np.empty((n_chan, 4, grid_n, grid_n), dtype=np.complex128)
    A = np.empty((n_chan, 4, grid_n, grid_n), dtype=np.float64) if want_abs else None
    if n_threads <= 0:
        n_threads = os.cpu_count() or 1
    used = _load().oracle_grid(uv.ctypes.data, freqs.ctypes.data, vis.ctypes.data, w_ptr, n_vis, n_chan,
                               grid_n, float(cell_du), support_W, oversample_O, table.ctypes.data,
                               G.ctypes.data, A.ctypes.data if want_abs else None, n_threads)
    return G, A, used


def grid_2d(uv, freqs, vis, weights, grid_n, cell_du, support_W, oversample_O, kernel_table_2d,
            want_abs: bool = True, n_threads: int = 0):
    """Gridding with a general 2-D complex kernel table [O+1, O+1, W, W] complex64 ([rv][ru][tv][tu]); SURVEY.md 8(f)-3.
    Returns (G complex128 [n_chan,4,N,N], A float64 or None, threads)."""
    uv, freqs = _np(uv, np.float64), _np(freqs, np.float64)
    vis = _np(vis, np.complex64)
    n_vis, n_chan = uv.shape[0], freqs.shape[0]
    assert vis.shape == (n_vis, n_chan, 4), vis.shape
    w_ptr = None
    if weights is not None:
        weights = _np(weights, np.float32)
        assert weights.shape == (n_vis, n_chan)
        w_ptr = weights.ctypes.data
    table = _np(kernel_table_2d, np.complex64)
    O1 = oversample_O + 1
    assert table.shape == (O1, O1, support_W, support_W), table.shape
    G = np.empty((n_chan, 4, grid_n, grid_n), dtype=np.complex128)
    A = np.empty((n_chan, 4, grid_n, grid_n), dtype=np.float64) if want_abs else None
    if n_threads <= 0:
        n_threads = os.cpu_count() or 1
    used = _load().oracle_grid_2d(uv.ctypes.data, freqs.ctypes.data, vis.ctypes.data, w_ptr, n_vis, n_chan,
                                  grid_n, float(cell_du), support_W, oversample_O, table.ctypes.data,
                                  G.ctypes.data, A.ctypes.data if want_abs else None, n_threads)
    return G, A, used
