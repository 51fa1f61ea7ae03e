"""Seeded synthetic magnetization fields for the five BASELINE.json configs.

This module serves both the CUDA path's tests/bench and the oracle's tests.  It
holds no arithmetic of the method (no tensor, no FFT convolution): it only
draws the inputs.  Recipe = SURVEY.md §8(d) / DESIGN.md "Input recipe".  The
paper's own benchmark inputs ("magnetization response to a
perpendicular magnetic field", scripts in the Boris repository) are not
available; these fields stand in for them.

Every generator returns M as float32 [3][nz][ny][nx] (x fastest), |M| = Ms in
every cell, drawn in fp64 from numpy.random.default_rng(seed) and rounded once.
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    hx: float
    hy: float
    hz: float
    Ms: float
    seed: int
    texture: str

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def h(self):
        return (self.hx, self.hy, self.hz)

    @property
    def cells(self):
        return self.nx * self.ny * self.nz


NM = 1e-9
CONFIGS = {
    "C1": Config("C1", 32, 32, 1, 5 * NM, 5 * NM, 3 * NM, 8.0e5, 1001, "random"),
    "C2": Config("C2", 256, 256, 1, 4 * NM, 4 * NM, 4 * NM, 8.6e5, 1002, "vortex"),
    "C3": Config("C3", 1024, 1024, 1, 2 * NM, 2 * NM, 1 * NM, 6.0e5, 1003, "domains"),
    "C4": Config("C4", 128, 128, 128, 2 * NM, 2 * NM, 2 * NM, 8.0e5, 1004, "random"),
    "C5": Config("C5", 512, 512, 32, 2 * NM, 2 * NM, 1 * NM, 1.1e6, 1005, "helix"),
}


def _normalise(m):
    return m / np.sqrt(np.sum(m * m, axis=0, keepdims=True))


def random_sphere(shape, rng):
    """Unit vectors uniform on the sphere: normalised N(0, I3) draws."""
    return _normalise(rng.standard_normal((3,) + tuple(shape)))


def vortex(shape, rng, core_radius=5.0, sigma=0.1):
    """In-plane counter-clockwise vortex, +z core exp(-(rho/5)^2), sigma=0.1 isotropic noise."""
    nz, ny, nx = shape
    y, x = np.meshgrid(np.arange(ny) - (ny - 1) / 2, np.arange(nx) - (nx - 1) / 2, indexing="ij")
    rho = np.sqrt(x * x + y * y)
    mz = np.exp(-(rho / core_radius) ** 2)
    inplane = np.sqrt(np.clip(1 - mz * mz, 0, None))
    safe = np.where(rho > 0, rho, 1.0)
    m = np.stack([-y / safe * inplane, x / safe * inplane, mz])
    m = np.broadcast_to(m[:, None], (3, nz, ny, nx)).copy()
    return _normalise(m + sigma * rng.standard_normal(m.shape))


def domains(shape, rng, fwhm=64.0, wall=0.1):
    """Up/down z-domains from a smoothed Gaussian field with Neel-like walls."""
    nz, ny, nx = shape
    sig = fwhm / 2.355
    g = rng.standard_normal((ny, nx))
    ky = np.fft.fftfreq(ny)[:, None]
    kx = np.fft.rfftfreq(nx)[None, :]
    filt = np.exp(-2 * (np.pi * sig) ** 2 * (kx * kx + ky * ky))   # periodic Gaussian blur
    g = np.fft.irfft2(np.fft.rfft2(g) * filt, s=(ny, nx))
    g = g / g.std()
    mz = np.tanh(g / wall)
    gy = (np.roll(g, -1, 0) - np.roll(g, 1, 0)) / 2
    gx = (np.roll(g, -1, 1) - np.roll(g, 1, 1)) / 2
    gn = np.sqrt(gx * gx + gy * gy)
    ux = np.where(gn > 0, gx / np.where(gn > 0, gn, 1), 1.0)
    uy = np.where(gn > 0, gy / np.where(gn > 0, gn, 1), 0.0)
    inplane = np.sqrt(np.clip(1 - mz * mz, 0, None))
    m = np.stack([inplane * ux, inplane * uy, mz])
    m = np.broadcast_to(m[:, None], (3, nz, ny, nx)).copy()
    return _normalise(m)


def helix(shape, rng, period=40.0, sigma=0.05):
    """Helix propagating along x: m = (0, cos, sin)(2 pi i / period) + 5 % noise."""
    nz, ny, nx = shape
    ph = 2 * np.pi * np.arange(nx) / period
    m = np.stack([np.zeros(nx), np.cos(ph), np.sin(ph)])
    m = np.broadcast_to(m[:, None, None, :], (3, nz, ny, nx)).copy()
    return _normalise(m + sigma * rng.standard_normal(m.shape))


_TEXTURES = {"random": random_sphere, "vortex": vortex, "domains": domains, "helix": helix}


def make_texture(texture, shape, Ms, seed):
    """M float32 [3][nz][ny][nx] for an arbitrary mesh shape (used by the small-mesh tests)."""
    rng = np.random.default_rng(seed)
    m = _TEXTURES[texture](tuple(shape), rng)
    return np.ascontiguousarray((Ms * m).astype(np.float32))


def make_input(cfg):
    """M for one of CONFIGS (pass the Config or its name)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    return make_texture(cfg.texture, cfg.shape, cfg.Ms, cfg.seed)


def sample_targets(shape, count=64, seed=0):
    """Target cells for sampled checks: 8 corners, face/edge/body centres, rest seeded-random."""
    nz, ny, nx = shape
    pts = []
    for k in sorted({0, nz // 2, nz - 1}):
        for j in sorted({0, ny // 2, ny - 1}):
            for i in sorted({0, nx // 2, nx - 1}):
                pts.append((k, j, i))
    rng = np.random.default_rng(seed)
    seen = set(pts)
    while len(pts) < count and len(seen) < nz * ny * nx:
        p = (int(rng.integers(nz)), int(rng.integers(ny)), int(rng.integers(nx)))
        if p not in seen:
            seen.add(p)
            pts.append(p)
    return pts[:count] if count < len(pts) else pts
