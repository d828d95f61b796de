"""Seeded synthetic input generators shared by the CPU oracle's tests and the CUDA path's tests/bench.
Holds no gridding arithmetic and imports neither `oracle` nor the CUDA binding."""
from .configs import CONFIGS, GridConfig, GridInputs, baseline_major, generate, scaled, C_LIGHT  # noqa: F401
from .pswf import make_kernel_table  # noqa: F401
