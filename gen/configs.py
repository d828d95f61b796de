"""Seeded synthetic MWA-shaped inputs for the five BASELINE.json configs (C1..C5).

No real MWA data, antenna layout or catalogue exists in this repository; these inputs stand in for
them with the paper's shapes: 512 antennas -> ~130,000 baselines, 768 channels, 4 polarisations
(PAPER.md:15).  The recipe is stated in DESIGN.md ("Input recipe").  This module holds
NONE of the gridding arithmetic: it produces (uv, freqs, vis, weights, du) and the kernel table,
which are handed unchanged to both the CUDA library and the CPU oracle.
"""
import math
from dataclasses import dataclass, replace

import torch

from . import rng
from .pswf import make_kernel_table

C_LIGHT = 299792458.0
BASE_SEED = 90200915


@dataclass(frozen=True)
class GridConfig:
    name: str
    index: int                 # k in BASELINE.json configs[k]; seed = BASE_SEED + k
    n_ant: int
    core_ant: int              # antennas drawn in the dense core disk (0 = single disk)
    core_radius_m: float
    radius_m: float
    n_int: int                 # integrations (earth rotation only when > 1)
    conjugates: bool
    n_chan: int
    f_lo_hz: float
    f_hi_hz: float
    grid_n: int
    support_W: int
    oversample_O: int
    n_src: int
    spectral_index: float      # S ~ (nu/nu_ref)^alpha ; 0 = flat
    random_weights: bool
    latitude_deg: float = -26.7
    dec_deg: float = -27.0
    int_seconds: float = 8.0

    @property
    def n_baselines(self) -> int:
        return self.n_ant * (self.n_ant - 1) // 2

    @property
    def n_vis(self) -> int:
        return self.n_baselines * self.n_int * (2 if self.conjugates else 1)

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    def freqs(self) -> torch.Tensor:
        if self.n_chan == 1:
            return torch.tensor([self.f_lo_hz], dtype=torch.float64)
        return torch.linspace(self.f_lo_hz, self.f_hi_hz, self.n_chan, dtype=torch.float64)

    # bytes that cross HBM once per call if nothing is re-read
    def algorithmic_bytes(self) -> int:
        nv, nc, n = self.n_vis, self.n_chan, self.grid_n
        return nv * nc * (32 + 4) + nv * 16 + nc * 8 + nc * 4 * n * n * 8

    def vis_pol(self) -> int:
        return self.n_vis * self.n_chan * 4

    def tap_updates(self) -> int:
        return self.vis_pol() * self.support_W ** 2


_C4_HALF_BAND = 0.5 * 767 * 40e3

CONFIGS = {
    "C1": GridConfig("C1", 0, 32, 0, 0.0, 1500.0, 1, True, 1, 150e6, 150e6, 256, 7, 8, 5, 0.0, False),
    "C2": GridConfig("C2", 1, 128, 0, 0.0, 1500.0, 1, True, 32, 140e6, 170e6, 1024, 7, 8, 20, 0.0, False),
    "C3": GridConfig("C3", 2, 512, 256, 300.0, 1500.0, 1, True, 1, 150e6, 150e6, 2048, 7, 8, 20, 0.0, False),
    "C4": GridConfig("C4", 3, 512, 256, 300.0, 1500.0, 1, False, 768, 155e6 - _C4_HALF_BAND,
                     155e6 + _C4_HALF_BAND, 1024, 7, 8, 20, -0.7, False),
    "C5": GridConfig("C5", 4, 512, 256, 300.0, 1500.0, 8, False, 64, 140e6, 170e6, 4096, 15, 16, 20, 0.0, True),
}


def scaled(cfg: GridConfig, **kw) -> GridConfig:
    """A config with some fields replaced (tests use smaller n_ant / n_chan / grid_n variants)."""
    return replace(cfg, **kw)


@dataclass
class GridInputs:
    cfg: GridConfig
    uv: torch.Tensor           # [n_vis, 2] f64 metres
    freqs: torch.Tensor        # [n_chan] f64 Hz
    vis: torch.Tensor          # [n_vis, n_chan, 4] complex64
    weights: torch.Tensor      # [n_vis, n_chan] f32
    cell_du: float             # wavelengths per cell
    kernel_table: torch.Tensor  # [O+1, W] f32 (CPU)
    sources: dict


def _disk(seed: int, stream: int, n: int, radius: float, first: int = 0) -> torch.Tensor:
    idx = torch.arange(first, first + n)
    r = radius * torch.sqrt(rng.uniform(seed, stream, idx))
    th = (2.0 * math.pi) * rng.uniform(seed, stream + 1, idx)
    return torch.stack([r * torch.cos(th), r * torch.sin(th)], dim=1)   # (east, north) metres


def antenna_positions(cfg: GridConfig) -> torch.Tensor:
    if cfg.core_ant > 0:
        core = _disk(cfg.seed, 10, cfg.core_ant, cfg.core_radius_m)
        rest = _disk(cfg.seed, 10, cfg.n_ant - cfg.core_ant, cfg.radius_m, first=cfg.core_ant)
        return torch.cat([core, rest], dim=0)
    return _disk(cfg.seed, 10, cfg.n_ant, cfg.radius_m)


def baseline_uv_metres(cfg: GridConfig) -> torch.Tensor:
    """[n_vis, 2] f64: rows ordered [integration][baseline], conjugate rows appended as a second half."""
    pos = antenna_positions(cfg)
    i, j = torch.triu_indices(cfg.n_ant, cfg.n_ant, offset=1)
    d = pos[j] - pos[i]                                   # (east, north)
    if cfg.n_int == 1:
        uv = d.clone()
    else:
        # textbook rotation, planar array: (X, Y, Z) = (-sin(lat) N, E, cos(lat) N); w discarded
        lat, dec = math.radians(cfg.latitude_deg), math.radians(cfg.dec_deg)
        X, Y, Z = -math.sin(lat) * d[:, 1], d[:, 0], math.cos(lat) * d[:, 1]
        rows = []
        for k in range(cfg.n_int):
            H = math.radians((k - 0.5 * (cfg.n_int - 1)) * cfg.int_seconds * (15.0 / 3600.0))
            u = math.sin(H) * X + math.cos(H) * Y
            v = -math.sin(dec) * math.cos(H) * X + math.sin(dec) * math.sin(H) * Y + math.cos(dec) * Z
            rows.append(torch.stack([u, v], dim=1))
        uv = torch.cat(rows, dim=0)
    if cfg.conjugates:
        uv = torch.cat([uv, -uv], dim=0)
    return uv.contiguous()


def cell_du(cfg: GridConfig, uv: torch.Tensor) -> float:
    """du such that the largest |u|,|v| (wavelengths, top channel) sits at 90% of the half grid."""
    s_max = float(cfg.freqs().max()) / C_LIGHT
    return float(uv.abs().max()) * s_max / (0.45 * cfg.grid_n)


def sky_model(cfg: GridConfig) -> dict:
    idx = torch.arange(cfg.n_src)
    l = 0.6 * rng.uniform(cfg.seed, 20, idx) - 0.3
    m = 0.6 * rng.uniform(cfg.seed, 21, idx) - 0.3
    a, b, g = 0.1 ** -0.8, 10.0 ** -0.8, -1.0 / 0.8       # inverse CDF of S^-1.8 on [0.1, 10]
    flux = (a - rng.uniform(cfg.seed, 22, idx) * (a - b)) ** g
    q = (0.2 * rng.uniform(cfg.seed, 23, idx) - 0.1) * flux
    u = (0.2 * rng.uniform(cfg.seed, 24, idx) - 0.1) * flux
    v = (0.2 * rng.uniform(cfg.seed, 25, idx) - 0.1) * flux
    # instrumental planes XX, XY, YX, YY
    bright = torch.stack([torch.complex(flux + q, torch.zeros_like(flux)), torch.complex(u, v),
                          torch.complex(u, -v), torch.complex(flux - q, torch.zeros_like(flux))], dim=1)
    return {"l": l, "m": m, "flux": flux, "brightness": bright}


def generate(cfg: GridConfig, device="cpu", rows_per_chunk: int = 0) -> GridInputs:
    """Build the inputs of one config on `device` (visibilities by direct sum in fp64)."""
    dev = torch.device(device)
    uv_cpu = baseline_uv_metres(cfg)
    du = cell_du(cfg, uv_cpu)
    freqs_cpu = cfg.freqs()
    sky = sky_model(cfg)
    n_base = cfg.n_vis // 2 if cfg.conjugates else cfg.n_vis
    nc, ns = cfg.n_chan, cfg.n_src

    uv = uv_cpu.to(dev)
    scale = (freqs_cpu / C_LIGHT).to(dev)                                   # [nc]
    spec = (freqs_cpu / 155e6) ** cfg.spectral_index if cfg.spectral_index else torch.ones(nc, dtype=torch.float64)
    bright = (spec[:, None, None] * sky["brightness"][None]).to(dev)        # [nc, ns, 4] c128
    l, m = sky["l"].to(dev), sky["m"].to(dev)

    vis = torch.empty((cfg.n_vis, nc, 4), dtype=torch.complex64, device=dev)
    if rows_per_chunk <= 0:
        rows_per_chunk = max(1, (1 << 22) // (nc * ns))
    for r0 in range(0, n_base, rows_per_chunk):
        r1 = min(n_base, r0 + rows_per_chunk)
        g = uv[r0:r1, 0:1] * l[None] + uv[r0:r1, 1:2] * m[None]              # [r, ns] metres
        ph = (-2.0 * math.pi) * scale[None, :, None] * g[:, None, :]        # [r, nc, ns]
        e = torch.polar(torch.ones_like(ph), ph)                            # c128
        v = torch.einsum("rcs,csp->rcp", e, bright)                         # [r, nc, 4]
        idx = (torch.arange(r0, r1, device=dev)[:, None, None] * nc
               + torch.arange(nc, device=dev)[None, :, None]) * 4 + torch.arange(4, device=dev)[None, None, :]
        noise = torch.complex(rng.normal(cfg.seed, 30, idx), rng.normal(cfg.seed, 31, idx)) * 0.01
        vis[r0:r1] = (v + noise).to(torch.complex64)
    if cfg.conjugates:
        vis[n_base:] = vis[:n_base].conj()

    if cfg.random_weights:
        w = torch.empty((cfg.n_vis, nc), dtype=torch.float32, device=dev)
        step = max(1, (1 << 24) // nc)
        for r0 in range(0, cfg.n_vis, step):
            r1 = min(cfg.n_vis, r0 + step)
            idx = torch.arange(r0, r1, device=dev)[:, None] * nc + torch.arange(nc, device=dev)[None, :]
            w[r0:r1] = (0.5 + rng.uniform(cfg.seed, 40, idx)).to(torch.float32)
    else:
        w = torch.ones((cfg.n_vis, nc), dtype=torch.float32, device=dev)

    table = torch.from_numpy(make_kernel_table(cfg.support_W, cfg.oversample_O))
    return GridInputs(cfg, uv, freqs_cpu.to(dev), vis, w, du, table, sky)


def baseline_major(g: GridInputs) -> GridInputs:
    """The same rows reordered [baseline][integration] (generated order is [integration][baseline]): consecutive rows are
    then the consecutive integrations of one baseline, 1 - 3.4 cells apart in C5 - the order a correlator dump in
    "baseline order" has and the one the register-ownership design (K3b) is made for.  No-op for a single integration."""
    cfg = g.cfg
    if cfg.n_int <= 1 or cfg.conjugates:
        return g
    nb = cfg.n_baselines
    idx = (torch.arange(cfg.n_int, device=g.uv.device)[None, :] * nb + torch.arange(nb, device=g.uv.device)[:, None]).reshape(-1)
    return GridInputs(cfg, g.uv[idx].contiguous(), g.freqs, g.vis[idx].contiguous(), g.weights[idx].contiguous(), g.cell_du,
                      g.kernel_table, g.sources)
