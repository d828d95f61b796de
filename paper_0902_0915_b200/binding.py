"""Thin ctypes binding of include/mwa_grid.h: argument marshalling only, same names as the C ABI.

Every step of the hot path runs in the CUDA library; there is no CPU fallback.  Importing this module
without the built library raises ImportError (build it with `python -m paper_0902_0915_b200._build`
or `__graft_entry__.build()`).
"""
import ctypes
import os

import torch

from . import _build

DESIGN_AUTO, DESIGN_ATOMIC, DESIGN_SMEM, DESIGN_ROMEIN, DESIGN_GATHER, DESIGN_CHAN, DESIGN_CHANWS, DESIGN_ROMEIN_SORTED = 0, 1, 2, 3, 4, 5, 6, 7
DESIGNS = {"auto": DESIGN_AUTO, "atomic": DESIGN_ATOMIC, "smem": DESIGN_SMEM, "romein": DESIGN_ROMEIN,
           "gather": DESIGN_GATHER, "chan": DESIGN_CHAN, "chanws": DESIGN_CHANWS, "romein_sorted": DESIGN_ROMEIN_SORTED}

if not os.path.exists(_build.LIB):
    raise ImportError(f"{_build.LIB} is missing: the CUDA library has not been built "
                      "(run `python -m paper_0902_0915_b200._build`); there is no CPU fallback")

_lib = ctypes.CDLL(_build.LIB)
_P, _I, _LL, _D = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong, ctypes.c_double

_lib.mwa_grid_plan_create.argtypes = [_I, _D, _I, _I, _P]
_lib.mwa_grid_plan_create.restype = _P
_lib.mwa_grid_plan_create_2d.argtypes = [_I, _D, _I, _I, _P]
_lib.mwa_grid_plan_create_2d.restype = _P
_lib.mwa_grid_plan_destroy.argtypes = [_P]
_lib.mwa_grid_plan_destroy.restype = None
_lib.mwa_grid_visibilities.argtypes = [_P, _P, _P, _P, _P, _LL, _I, _P, _P]
_lib.mwa_grid_visibilities.restype = _I
_lib.mwa_grid_visibilities_host.argtypes = [_P, _P, _P, _P, _P, _LL, _I, _P, _P]
_lib.mwa_grid_visibilities_host.restype = _I
_lib.mwa_grid_visibilities_noalloc.argtypes = [_I, _D, _I, _I, _P, _P, _P, _P, _P, _LL, _I, _P, _P]
_lib.mwa_grid_visibilities_noalloc.restype = _I
_lib.mwa_grid_compute_indices.argtypes = [_P, _P, _P, _LL, _I, _P, _P]
_lib.mwa_grid_compute_indices.restype = _I
_lib.mwa_grid_weights_grid.argtypes = [_P, _P, _P, _P, _LL, _I, _P, _P]
_lib.mwa_grid_weights_grid.restype = _I
_lib.mwa_grid_count_dropped.argtypes = [_P, _P, _P, _LL, _I, _P, _P]
_lib.mwa_grid_count_dropped.restype = _I
_lib.mwa_grid_plan_set_mfs.argtypes = [_P, _I]
_lib.mwa_grid_plan_set_mfs.restype = _I
_lib.mwa_grid_plan_set_accumulate.argtypes = [_P, _I]
_lib.mwa_grid_plan_set_accumulate.restype = _I
_lib.mwa_grid_plan_set_design.argtypes = [_P, _I]
_lib.mwa_grid_plan_set_design.restype = _I
_lib.mwa_grid_plan_set_profiling.argtypes = [_P, _I]
_lib.mwa_grid_plan_set_profiling.restype = _I
_lib.mwa_grid_plan_stage_ms.argtypes = [_P, _P, _I]
_lib.mwa_grid_plan_stage_ms.restype = _I
_lib.mwa_grid_plan_last_launches.argtypes = [_P]
_lib.mwa_grid_plan_last_launches.restype = _I
_lib.mwa_grid_plan_last_design.argtypes = [_P]
_lib.mwa_grid_plan_last_design.restype = _I
_lib.mwa_grid_plan_set_list_pool.argtypes = [_P, _LL]
_lib.mwa_grid_plan_set_list_pool.restype = _I
_lib.mwa_grid_plan_last_stats.argtypes = [_P, _P, _I]
_lib.mwa_grid_plan_last_stats.restype = _I
_lib.mwa_grid_probe_fp32.argtypes = [_P, _P, _P]
_lib.mwa_grid_probe_fp32.restype = _I
_lib.mwa_image_from_grid.argtypes = [_P, _P, _P, _LL, _P]
_lib.mwa_image_from_grid.restype = _I
_lib.mwa_image_stokes.argtypes = [_P, _P, _P, _P, _I, _P]
_lib.mwa_image_stokes.restype = _I
_lib.mwa_image_correction.argtypes = [_P, _P, _I]
_lib.mwa_image_correction.restype = _I
_lib.mwa_grid_probe_smem_atomics.argtypes = [_P, _P, _P]
_lib.mwa_grid_probe_smem_atomics.restype = _I
_lib.mwa_grid_last_error.argtypes = []
_lib.mwa_grid_last_error.restype = ctypes.c_char_p

EXPORTS = ["mwa_grid_plan_create", "mwa_grid_plan_destroy", "mwa_grid_visibilities", "mwa_grid_visibilities_host",
           "mwa_grid_compute_indices", "mwa_grid_plan_set_design", "mwa_grid_plan_set_profiling",
           "mwa_grid_plan_stage_ms", "mwa_grid_plan_last_launches", "mwa_grid_plan_last_design", "mwa_grid_plan_last_stats", "mwa_grid_plan_set_list_pool", "mwa_grid_probe_fp32", "mwa_grid_last_error",
           "mwa_image_from_grid", "mwa_image_correction", "mwa_image_stokes", "mwa_grid_probe_smem_atomics", "mwa_grid_count_dropped", "mwa_grid_plan_set_accumulate", "mwa_grid_plan_set_mfs", "mwa_grid_weights_grid", "mwa_grid_plan_create_2d",
           "mwa_grid_visibilities_noalloc"]


class MwaGridError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"mwa_grid error {code}: {msg}")
        self.code = code


def mwa_grid_last_error() -> str:
    return _lib.mwa_grid_last_error().decode()


def _check(rc: int) -> int:
    if rc < 0:
        raise MwaGridError(rc, mwa_grid_last_error())
    return rc


def _ptr(t, dtype, device_type, name):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor):
        raise TypeError(f"{name} must be a torch.Tensor")
    if t.dtype != dtype:
        raise TypeError(f"{name} must be {dtype}, got {t.dtype}")
    if t.device.type != device_type:
        raise ValueError(f"{name} must live on {device_type}, got {t.device}")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    return t.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def mwa_grid_plan_create(grid_n: int, cell_du: float, support_W: int, oversample_O: int, kernel_table) -> int:
    """kernel_table: CPU float32 tensor / array of shape [O+1, W].  Returns the opaque plan handle."""
    tab = torch.as_tensor(kernel_table, dtype=torch.float32, device="cpu").contiguous()
    if tab.numel() != (int(oversample_O) + 1) * int(support_W):
        raise ValueError("kernel_table must hold (O+1)*W floats")
    h = _lib.mwa_grid_plan_create(int(grid_n), float(cell_du), int(support_W), int(oversample_O), tab.data_ptr())
    if not h:
        raise MwaGridError(-1, mwa_grid_last_error())
    return h


def mwa_grid_plan_create_2d(grid_n: int, cell_du: float, support_W: int, oversample_O: int, kernel_table_2d) -> int:
    """kernel_table_2d: CPU complex64 tensor / array of shape [O+1, O+1, W, W] ([rv][ru][tv][tu]).  Returns the plan handle."""
    tab = torch.as_tensor(kernel_table_2d, dtype=torch.complex64, device="cpu").contiguous()
    if tuple(tab.shape) != (int(oversample_O) + 1, int(oversample_O) + 1, int(support_W), int(support_W)):
        raise ValueError("kernel_table_2d must be complex64 [O+1, O+1, W, W]")
    h = _lib.mwa_grid_plan_create_2d(int(grid_n), float(cell_du), int(support_W), int(oversample_O), tab.data_ptr())
    if not h:
        raise MwaGridError(-1, mwa_grid_last_error())
    return h


def mwa_grid_plan_destroy(plan) -> None:
    if plan:
        _lib.mwa_grid_plan_destroy(plan)


def mwa_grid_visibilities(plan, uv_f64, freqs, vis_c64, weights, n_vis, n_chan, grid_out, stream=None) -> None:
    """Device tensors: uv f64 [n_vis,2], freqs f64 [n_chan], vis complex64 [n_vis,n_chan,4],
    weights f32 [n_vis,n_chan] or None, grid_out complex64 [n_chan,4,N,N] (overwritten).  Asynchronous."""
    _check(_lib.mwa_grid_visibilities(plan, _ptr(uv_f64, torch.float64, "cuda", "uv_f64"),
                                      _ptr(freqs, torch.float64, "cuda", "freqs"),
                                      _ptr(vis_c64, torch.complex64, "cuda", "vis_c64"),
                                      _ptr(weights, torch.float32, "cuda", "weights"),
                                      int(n_vis), int(n_chan), _ptr(grid_out, torch.complex64, "cuda", "grid_out"),
                                      _stream_ptr(stream)))


def mwa_grid_visibilities_host(plan, uv_f64, freqs, vis_c64, weights, n_vis, n_chan, grid_out, stream=None) -> None:
    """The same call on HOST tensors (pinned for full PCIe speed); synchronises before returning."""
    _check(_lib.mwa_grid_visibilities_host(plan, _ptr(uv_f64, torch.float64, "cpu", "uv_f64"),
                                           _ptr(freqs, torch.float64, "cpu", "freqs"),
                                           _ptr(vis_c64, torch.complex64, "cpu", "vis_c64"),
                                           _ptr(weights, torch.float32, "cpu", "weights"),
                                           int(n_vis), int(n_chan), _ptr(grid_out, torch.complex64, "cpu", "grid_out"),
                                           _stream_ptr(stream)))


NOALLOC_MAX_VIS, NOALLOC_MAX_CHAN, NOALLOC_MAX_GRID_N = 131072, 1024, 2048      # MWA_GRID_NOALLOC_MAX_* of the header


def mwa_grid_visibilities_noalloc(grid_n, cell_du, support_W, oversample_O, kernel_table_dev, uv_f64, freqs, vis_c64, weights,
                                  n_vis, n_chan, grid_out, stream=None) -> None:
    """The gridding call that allocates nothing (no plan; GATHER design on a static device scratch array of the library).
    kernel_table_dev: DEVICE float32 [O+1, W]; the other tensors as in mwa_grid_visibilities.  Limits: NOALLOC_MAX_*.
    Calls that overlap on the GPU race on the shared scratch.  Asynchronous."""
    if kernel_table_dev is not None and kernel_table_dev.numel() != (int(oversample_O) + 1) * int(support_W):
        raise ValueError("kernel_table_dev must hold (O+1)*W floats")
    _check(_lib.mwa_grid_visibilities_noalloc(int(grid_n), float(cell_du), int(support_W), int(oversample_O),
                                              _ptr(kernel_table_dev, torch.float32, "cuda", "kernel_table_dev"),
                                              _ptr(uv_f64, torch.float64, "cuda", "uv_f64"),
                                              _ptr(freqs, torch.float64, "cuda", "freqs"),
                                              _ptr(vis_c64, torch.complex64, "cuda", "vis_c64"),
                                              _ptr(weights, torch.float32, "cuda", "weights"),
                                              int(n_vis), int(n_chan), _ptr(grid_out, torch.complex64, "cuda", "grid_out"),
                                              _stream_ptr(stream)))


def mwa_grid_compute_indices(plan, uv_f64, freqs, n_vis, n_chan, out_idx, stream=None) -> None:
    """out_idx: device int32 [n_vis, n_chan, 4] = (iu, iv, ru, rv) or -1s."""
    _check(_lib.mwa_grid_compute_indices(plan, _ptr(uv_f64, torch.float64, "cuda", "uv_f64"),
                                         _ptr(freqs, torch.float64, "cuda", "freqs"), int(n_vis), int(n_chan),
                                         _ptr(out_idx, torch.int32, "cuda", "out_idx"), _stream_ptr(stream)))


def mwa_grid_weights_grid(plan, uv_f64, freqs, weights, n_vis, n_chan, wgrid_out, stream=None) -> None:
    """f3: companion weights grid, float32 [n_chan, N, N] = sum of tap * weight per cell."""
    _check(_lib.mwa_grid_weights_grid(plan, _ptr(uv_f64, torch.float64, "cuda", "uv_f64"), _ptr(freqs, torch.float64, "cuda", "freqs"),
                                      _ptr(weights, torch.float32, "cuda", "weights"), int(n_vis), int(n_chan),
                                      _ptr(wgrid_out, torch.float32, "cuda", "wgrid_out"), _stream_ptr(stream)))


def mwa_grid_count_dropped(plan, uv_f64, freqs, n_vis, n_chan, stream=None) -> int:
    """Number of (row, channel) samples the gridder drops (R11) for these coordinates.  Synchronises."""
    out = ctypes.c_longlong(0)
    _check(_lib.mwa_grid_count_dropped(plan, _ptr(uv_f64, torch.float64, "cuda", "uv_f64"),
                                       _ptr(freqs, torch.float64, "cuda", "freqs"), int(n_vis), int(n_chan),
                                       ctypes.cast(ctypes.pointer(out), ctypes.c_void_p), _stream_ptr(stream)))
    return int(out.value)


def mwa_grid_plan_set_mfs(plan, enabled: bool) -> None:
    """f3: multi-frequency synthesis - all channels of a call are summed onto one grid [4, N, N]."""
    _check(_lib.mwa_grid_plan_set_mfs(plan, 1 if enabled else 0))


def mwa_grid_plan_set_accumulate(plan, enabled: bool) -> None:
    """f3: grid_out += gridded samples instead of grid_out = (cells nothing reaches stay as they are)."""
    _check(_lib.mwa_grid_plan_set_accumulate(plan, 1 if enabled else 0))


def mwa_grid_plan_set_design(plan, design) -> None:
    _check(_lib.mwa_grid_plan_set_design(plan, DESIGNS[design] if isinstance(design, str) else int(design)))


def mwa_grid_plan_set_profiling(plan, enabled: bool) -> None:
    _check(_lib.mwa_grid_plan_set_profiling(plan, 1 if enabled else 0))


def mwa_grid_plan_stage_ms(plan):
    """(binning_ms, gridding_ms, total_ms) of the last profiled call."""
    buf = (ctypes.c_float * 3)()
    _check(_lib.mwa_grid_plan_stage_ms(plan, ctypes.cast(buf, ctypes.c_void_p), 3))
    return tuple(float(x) for x in buf)


def mwa_grid_plan_last_launches(plan) -> int:
    return int(_lib.mwa_grid_plan_last_launches(plan))


def mwa_grid_plan_last_design(plan) -> str:
    """Name of the design the last gridding call ran (resolves AUTO; synchronises)."""
    code = _check(_lib.mwa_grid_plan_last_design(plan))
    return {v: k for k, v in DESIGNS.items()}[code]


def mwa_grid_plan_last_stats(plan):
    """Counters of the last K6 call: dict(error, items, items_with_hits, batches, max_hits, swept_items).  Synchronises."""
    buf = (ctypes.c_longlong * 32)()
    _check(_lib.mwa_grid_plan_last_stats(plan, ctypes.cast(buf, ctypes.c_void_p), 32))
    return {"error": int(buf[0]), "items": int(buf[1]), "items_with_hits": int(buf[2]), "batches": int(buf[3]),
            "max_hits": int(buf[4]), "swept_items": int(buf[5]), "k5_dense_items": int(buf[6]), "timing": [int(x) for x in buf[8:32]],
            "k3c_heavy_items": int(buf[31])}


def mwa_grid_probe_smem_atomics(plan, stream=None) -> float:
    """Conflict-free red.shared.add.f32 lane-atomics per second of the whole device (measurement utility)."""
    buf = (ctypes.c_double * 1)()
    _check(_lib.mwa_grid_probe_smem_atomics(plan, ctypes.cast(buf, ctypes.c_void_p), _stream_ptr(stream)))
    return float(buf[0])


def mwa_grid_plan_set_list_pool(plan, entries: int) -> None:
    """Diagnostics: cap K6's hit-list pool (0 = default); overflowing items take the in-kernel sweep."""
    _check(_lib.mwa_grid_plan_set_list_pool(plan, int(entries)))


def mwa_image_from_grid(plan, grid, image, n_planes, stream=None) -> None:
    """f1: corrected dirty images of `n_planes` N x N uv grids (device complex64); `image` may be `grid` (in place)."""
    _check(_lib.mwa_image_from_grid(plan, _ptr(grid, torch.complex64, "cuda", "grid"),
                                    _ptr(image, torch.complex64, "cuda", "image"), int(n_planes), _stream_ptr(stream)))


def mwa_image_stokes(plan, image, matrix, stokes_out, n_chan, stream=None) -> None:
    """f2: stokes_out[c, k] = sum_j matrix[..., k, j] * image[c, j]; matrix complex64 [N, N, 4, 4]; in place allowed."""
    _check(_lib.mwa_image_stokes(plan, _ptr(image, torch.complex64, "cuda", "image"),
                                 _ptr(matrix, torch.complex64, "cuda", "matrix"),
                                 _ptr(stokes_out, torch.complex64, "cuda", "stokes_out"), int(n_chan), _stream_ptr(stream)))


def mwa_image_correction(plan, n: int):
    """The plan's correction function c^(p' - N/2), p' = 0..n-1, as a float64 CPU tensor."""
    out = torch.empty(int(n), dtype=torch.float64)
    k = _check(_lib.mwa_image_correction(plan, out.data_ptr(), int(n)))
    return out[:k]


def mwa_grid_probe_fp32(plan, stream=None):
    """(TFLOP/s of fma.rn.f32, TFLOP/s of fma.rn.f32x2) measured with a register-only loop."""
    buf = (ctypes.c_double * 2)()
    _check(_lib.mwa_grid_probe_fp32(plan, ctypes.cast(buf, ctypes.c_void_p), _stream_ptr(stream)))
    return float(buf[0]), float(buf[1])


class Plan:
    """Owns a plan handle; `grid()` allocates the output on the inputs' device and calls the ABI."""

    def __init__(self, grid_n, cell_du, support_W, oversample_O, kernel_table, design="auto", table_2d=False):
        self.grid_n, self.support_W, self.oversample_O = int(grid_n), int(support_W), int(oversample_O)
        self.mfs = False
        create = mwa_grid_plan_create_2d if table_2d else mwa_grid_plan_create
        self.handle = create(grid_n, cell_du, support_W, oversample_O, kernel_table)
        if design != "auto":
            mwa_grid_plan_set_design(self.handle, design)

    def set_mfs(self, enabled: bool):
        mwa_grid_plan_set_mfs(self.handle, enabled)
        self.mfs = bool(enabled)

    def set_design(self, design):
        mwa_grid_plan_set_design(self.handle, design)

    def grid(self, uv, freqs, vis, weights=None, out=None, stream=None):
        n_vis, n_chan = int(uv.shape[0]), int(freqs.shape[0])
        # the C ABI takes bare pointers and sizes: a wrong shape or device here would read or write out of bounds
        if tuple(uv.shape) != (n_vis, 2):
            raise ValueError(f"uv must be [n_vis, 2], got {tuple(uv.shape)}")
        if vis is not None and tuple(vis.shape) != (n_vis, n_chan, 4):
            raise ValueError(f"vis must be [n_vis={n_vis}, n_chan={n_chan}, 4], got {tuple(vis.shape)}")
        if weights is not None and tuple(weights.shape) != (n_vis, n_chan):
            raise ValueError(f"weights must be [n_vis={n_vis}, n_chan={n_chan}], got {tuple(weights.shape)}")
        if out is None:
            out = torch.empty((1 if self.mfs else n_chan, 4, self.grid_n, self.grid_n), dtype=torch.complex64, device=uv.device)
        elif tuple(out.shape) != (1 if self.mfs else n_chan, 4, self.grid_n, self.grid_n):
            raise ValueError(f"out must be [{'1' if self.mfs else n_chan}, 4, {self.grid_n}, {self.grid_n}], got {tuple(out.shape)}")
        for name, t in (("freqs", freqs), ("vis", vis), ("weights", weights), ("out", out)):
            if t is not None and t.device != uv.device:
                raise ValueError(f"{name} lives on {t.device}, uv on {uv.device}: all arguments must be on the plan's device")
        mwa_grid_visibilities(self.handle, uv, freqs, vis, weights, n_vis, n_chan, out, stream)
        return out

    def image(self, grid, out=None, stream=None):
        """Corrected dirty images of the grids of `grid` [..., N, N]; in place when out is grid."""
        if out is None:
            out = torch.empty_like(grid)
        mwa_image_from_grid(self.handle, grid, out, grid.numel() // (self.grid_n * self.grid_n), stream)
        return out

    def stokes(self, image, matrix, out=None, stream=None):
        """Stokes conversion of [n_chan, 4, N, N] images with a [N, N, 4, 4] matrix field; in place when out is image."""
        if tuple(matrix.shape) != (self.grid_n, self.grid_n, 4, 4) or tuple(image.shape[1:]) != (4, self.grid_n, self.grid_n):
            raise ValueError("image must be [n_chan, 4, N, N] and matrix [N, N, 4, 4]")
        if out is None:
            out = torch.empty_like(image)
        mwa_image_stokes(self.handle, image, matrix, out, int(image.shape[0]), stream)
        return out

    def indices(self, uv, freqs, stream=None):
        n_vis, n_chan = int(uv.shape[0]), int(freqs.shape[0])
        out = torch.empty((n_vis, n_chan, 4), dtype=torch.int32, device=uv.device)
        mwa_grid_compute_indices(self.handle, uv, freqs, n_vis, n_chan, out, stream)
        return out

    def close(self):
        if self.handle:
            mwa_grid_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
