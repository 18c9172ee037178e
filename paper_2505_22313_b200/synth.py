"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module holds NONE of the method's arithmetic (no phase, no DFT of a field, no transfer
function): it only manufactures height maps `h` (fp32, metres) and target intensities `T`
(fp32).  It is the one module that serves both sides: tests and bench.py generate an array ONCE
here and hand the same bytes to the CUDA library and (after download) to the fp64 oracle, so
parity never depends on two generators agreeing.

Every array is a pure function of (seed, stream_id, linear index) through an integer
counter-based mix (murmur3 finaliser on 32-bit lanes, done in int64 so it is bit-identical on
CPU and CUDA), mapped to U = k * 2^-24 in [0, 1).  Seeds: 20250522 + config index;
stream 0 = height, 1 = target (2, 3 = second Box-Muller uniforms).

They stand in for data the paper used and did not publish: randomly initialised height maps
(PAPER.md:141), low-pass calibration patterns, quantised 10-bit layouts
(PAPER.md:153), hologram target images.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional, Tuple

import torch

_M32 = 0xFFFFFFFF
_CHUNK = 1 << 25  # elements per generation chunk (bounds temporaries to ~1.5 GiB on the GPU)


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json configuration made concrete."""
    name: str
    index: int
    ny: int
    nx: int
    pitch: float
    lambdas: Tuple[float, ...]
    n_refr: Tuple[float, ...]
    z: float
    sigma_px: float = 0.0          # Gaussian pre-filter (config 3)
    write_intensity: bool = False  # config 4: "intensity-only output plus L2 loss gradient"
    height_kind: str = "uniform"   # uniform | blur | gray256 | lattice
    h_max: float = 1.1e-6
    target_kind: str = "uniform"   # uniform | blur | lattice

    @property
    def seed(self) -> int:
        return 20250522 + self.index

    @property
    def points(self) -> int:
        return self.ny * self.nx * len(self.lambdas)

    def scaled(self, ny: int, nx: int) -> "Config":
        """Same recipe and optics on a smaller grid (parity-test sizes)."""
        return dataclasses.replace(self, ny=ny, nx=nx, name=f"{self.name}@{ny}x{nx}")


CONFIGS = {
    "C1": Config("C1", 0, 1024, 1024, 1.0e-6, (532e-9,), (1.46,), 1.0e-3,
                 height_kind="uniform", h_max=532e-9 / 0.46, target_kind="uniform"),
    "C2": Config("C2", 1, 8192, 8192, 0.5e-6, (450e-9, 550e-9, 650e-9), (1.5, 1.5, 1.5), 20e-3,
                 height_kind="blur", h_max=1.2e-6, target_kind="blur"),
    "C3": Config("C3", 2, 16384, 16384, 0.25e-6, (550e-9,), (1.5,), 10e-3, sigma_px=3.0,
                 height_kind="gray256", h_max=1.1e-6, target_kind="blur"),
    "C4": Config("C4", 3, 65536, 65536, 0.25e-6, (550e-9,), (1.5,), 50e-3,
                 write_intensity=True, height_kind="uniform", h_max=1.1e-6,
                 target_kind="lattice"),
    "C5": Config("C5", 4, 98304, 65536, 0.25e-6, (550e-9,), (1.5,), 100e-3,
                 height_kind="lattice", h_max=1.1e-6, target_kind="lattice"),
}


# --------------------------------------------------------------------------------------------
# counter-based uniform generator
# --------------------------------------------------------------------------------------------
def _fmix32(x: torch.Tensor) -> torch.Tensor:
    x = x ^ (x >> 16)
    x = (x * 0x85EBCA6B) & _M32
    x = x ^ (x >> 13)
    x = (x * 0xC2B2AE35) & _M32
    x = x ^ (x >> 16)
    return x


def hash_u01(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """U = k * 2^-24, k the top 24 bits of a 32-bit mix of (seed, stream, 64-bit index).
    `index` is an int64 tensor (any shape); returns fp32 of the same shape."""
    lo = index & _M32
    hi = (index >> 32) & _M32
    key = (seed * 0x9E3779B1 + stream * 0x7F4A7C15 + 0x632BE5AB) & _M32
    x = _fmix32(lo ^ key)
    x = _fmix32((x + hi * 0x9E3779B9 + 0x165667B1) & _M32)
    return (x >> 8).to(torch.float32) * (1.0 / 16777216.0)


def uniform_plane(seed: int, stream: int, ny: int, nx: int, device, scale: float = 1.0,
                  out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """[ny, nx] fp32 plane of hash_u01 over the row-major linear index, times `scale`
    (one fp32 multiply)."""
    n = ny * nx
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=device)
    flat = out.view(-1)
    s = torch.tensor(scale, dtype=torch.float32, device=device)
    for start in range(0, n, _CHUNK):
        stop = min(n, start + _CHUNK)
        idx = torch.arange(start, stop, dtype=torch.int64, device=device)
        flat[start:stop] = hash_u01(seed, stream, idx) * s
    return out.view(ny, nx)


def gray256_plane(seed: int, stream: int, ny: int, nx: int, device, h_max: float) -> torch.Tensor:
    """round(U * 255) * (h_max / 255): 256 gray levels (config 3)."""
    n = ny * nx
    out = torch.empty(n, dtype=torch.float32, device=device)
    step = torch.tensor(h_max / 255.0, dtype=torch.float32, device=device)
    for start in range(0, n, _CHUNK):
        stop = min(n, start + _CHUNK)
        idx = torch.arange(start, stop, dtype=torch.int64, device=device)
        out[start:stop] = torch.round(hash_u01(seed, stream, idx) * 255.0) * step
    return out.view(ny, nx)


def blurred_noise_plane(seed: int, stream: int, ny: int, nx: int, device, sigma_px: float,
                        lo: float, hi: float) -> torch.Tensor:
    """Box-Muller normal from two hashed uniforms -> periodic Gaussian blur (sigma_px) -> affine
    rescale so min -> lo, max -> hi (configs 2, 3).  The blur is input manufacture, done with
    torch.fft on whatever device the plane lives on."""
    u1 = uniform_plane(seed, stream, ny, nx, device)
    u2 = uniform_plane(seed, stream + 2, ny, nx, device)
    g = torch.sqrt(-2.0 * torch.log(1.0 - u1)) * torch.cos((2.0 * math.pi) * u2)
    del u1, u2
    ky = torch.fft.fftfreq(ny, device=device, dtype=torch.float32)
    kx = torch.fft.rfftfreq(nx, device=device, dtype=torch.float32)
    c = -2.0 * math.pi ** 2 * sigma_px ** 2
    spec = torch.fft.rfft2(g)
    del g
    spec *= torch.exp(c * ky * ky)[:, None]
    spec *= torch.exp(c * kx * kx)[None, :]
    g = torch.fft.irfft2(spec, s=(ny, nx))
    del spec
    mn, mx = g.min(), g.max()
    g = (g - mn) * ((hi - lo) / (mx - mn)) + lo
    return g.clamp_(lo, hi).to(torch.float32).contiguous()


def lattice_plane(seed: int, stream: int, ny: int, nx: int, device, cell: int, scale: float,
                  smooth: bool) -> torch.Tensor:
    """Per-point computable smooth field: interpolation of a hashed U lattice with `cell`-pixel
    cells (periodic), bilinear (smooth=False, config 4/5 target) or cubic-Hermite "smoothstep"
    weights (smooth=True, config 5 height); times `scale`.  Range [0, scale) by construction."""
    cy, cx = max(1, ny // cell), max(1, nx // cell)
    lat = uniform_plane(seed, stream, cy, cx, device)
    out = torch.empty((ny, nx), dtype=torch.float32, device=device)
    xs = torch.arange(nx, device=device)
    ix0 = (xs // cell) % cx
    ix1 = (ix0 + 1) % cx
    tx = (xs % cell).to(torch.float32) / float(cell)
    if smooth:
        tx = tx * tx * (3.0 - 2.0 * tx)
    rows = max(1, _CHUNK // nx)
    for y0 in range(0, ny, rows):
        y1 = min(ny, y0 + rows)
        ys = torch.arange(y0, y1, device=device)
        iy0 = (ys // cell) % cy
        iy1 = (iy0 + 1) % cy
        ty = (ys % cell).to(torch.float32) / float(cell)
        if smooth:
            ty = ty * ty * (3.0 - 2.0 * ty)
        a = lat[iy0][:, ix0] * (1.0 - tx) + lat[iy0][:, ix1] * tx
        b = lat[iy1][:, ix0] * (1.0 - tx) + lat[iy1][:, ix1] * tx
        out[y0:y1] = (a * (1.0 - ty[:, None]) + b * ty[:, None]) * scale
    return out


# --------------------------------------------------------------------------------------------
# per-config recipes
# --------------------------------------------------------------------------------------------
def make_height(cfg: Config, device="cpu") -> torch.Tensor:
    """fp32 [ny, nx] height map in metres, per SURVEY.md section 8(d)."""
    if cfg.height_kind == "uniform":
        return uniform_plane(cfg.seed, 0, cfg.ny, cfg.nx, device, scale=cfg.h_max)
    if cfg.height_kind == "blur":
        return blurred_noise_plane(cfg.seed, 0, cfg.ny, cfg.nx, device, 4.0, 0.0, cfg.h_max)
    if cfg.height_kind == "gray256":
        return gray256_plane(cfg.seed, 0, cfg.ny, cfg.nx, device, cfg.h_max)
    if cfg.height_kind == "lattice":
        return lattice_plane(cfg.seed, 0, cfg.ny, cfg.nx, device, 16, cfg.h_max, smooth=True)
    raise ValueError(cfg.height_kind)


def make_target(cfg: Config, device="cpu") -> torch.Tensor:
    """fp32 [ny, nx] target intensity (one target shared by all wavelengths)."""
    if cfg.target_kind == "uniform":
        return uniform_plane(cfg.seed, 1, cfg.ny, cfg.nx, device)
    if cfg.target_kind == "blur":
        return blurred_noise_plane(cfg.seed, 1, cfg.ny, cfg.nx, device, 8.0, 0.0, 2.0)
    if cfg.target_kind == "lattice":
        return lattice_plane(cfg.seed, 1, cfg.ny, cfg.nx, device, 64, 2.0, smooth=False)
    raise ValueError(cfg.target_kind)


def tile_plane(small: torch.Tensor, ry: int, rx: int) -> torch.Tensor:
    """Periodic tiling (pin P-k): [py, px] -> [ry*py, rx*px]."""
    return small.repeat(ry, rx).contiguous()
