"""Synthetic kappa / S fields for the five BASELINE.json configs (recipe: DESIGN.md "Input recipe").

The paper's own workloads are its photo-ionisation tests (128^3, N_side = 8) and
its timing runs (64^3/128^3/256^3 with N_side = 4/8/16).  Their fields come from a
chemistry solver that is not available, so seeded synthetic fields with the shapes and optical-depth
ranges BASELINE.json prescribes stand in for them.

All arrays are produced in fp64, cast to fp32 once, shape [nbins][nz][ny][nx] (x fastest).
kappa is per cell width (cell_width = 1), boundary inflow is zero, one ray per cell (r = 1).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class ConfigSpec:
    name: str
    dims: tuple          # (nx, ny, nz)
    nside: int
    nbins: int
    seed: int
    kind: str            # "uniform" | "lognormal" | "bubbles"
    sigma: float = 1.0
    nbubbles: int = 0
    clip: tuple | None = None
    nu: tuple = (1.0,)

    @property
    def ndirs(self) -> int:
        return 12 * self.nside * self.nside

    @property
    def ncell(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2]


CONFIGS = {
    "C1": ConfigSpec("C1", (32, 32, 32), 2, 1, 0, "uniform"),
    "C2": ConfigSpec("C2", (64, 64, 64), 8, 1, 1, "lognormal", sigma=1.0),
    "C3": ConfigSpec("C3", (128, 128, 128), 16, 1, 2, "bubbles", sigma=1.0, nbubbles=8),
    "C4": ConfigSpec("C4", (256, 256, 256), 16, 1, 3, "bubbles", sigma=1.5, nbubbles=64, clip=(1e-4, 1e2)),
    "C5": ConfigSpec("C5", (128, 128, 512), 16, 3, 4, "bubbles", sigma=1.5, nbubbles=64, clip=(1e-4, 1e2),
                     nu=(1.0, 1.5, 2.5)),
}


def config_spec(name: str) -> ConfigSpec:
    return CONFIGS[name]


def _gaussian_field(rng, dims):
    """Zero-mean unit-variance Gaussian random field with P(k) ~ k^-3, shape (nz, ny, nx)."""
    nx, ny, nz = dims
    white = rng.standard_normal((nz, ny, nx))
    fk = np.fft.rfftn(white, axes=(0, 1, 2))
    kz = 2.0 * np.pi * np.fft.fftfreq(nz)[:, None, None]
    ky = 2.0 * np.pi * np.fft.fftfreq(ny)[None, :, None]
    kx = 2.0 * np.pi * np.fft.rfftfreq(nx)[None, None, :]
    k2 = kx * kx + ky * ky + kz * kz
    k2[0, 0, 0] = 1.0
    amp = k2 ** (-0.75)                     # sqrt(P) = k^-3/2
    amp[0, 0, 0] = 0.0
    fk *= amp
    del amp, k2
    g = np.fft.irfftn(fk, s=(nz, ny, nx), axes=(0, 1, 2))
    del fk
    g -= g.mean()
    g /= g.std()
    return g


def _bubble_xhi(rng, dims, nbubbles):
    """Neutral fraction: 1e-4 inside seeded spherical bubbles (radius 6-20 cells), 1 outside, tanh edge."""
    nx, ny, nz = dims
    centres = rng.uniform(0.0, 1.0, size=(nbubbles, 3)) * np.array([nx, ny, nz], dtype=np.float64)
    radii = rng.uniform(6.0, 20.0, size=nbubbles)
    z = (np.arange(nz, dtype=np.float64) + 0.5)[:, None, None]
    y = (np.arange(ny, dtype=np.float64) + 0.5)[None, :, None]
    x = (np.arange(nx, dtype=np.float64) + 0.5)[None, None, :]
    xhi = np.ones((nz, ny, nx), dtype=np.float64)
    for (cx, cy, cz), R in zip(centres, radii):
        # only touch the bounding box of the bubble (+ a few edge widths)
        pad = R + 8.0
        z0, z1 = max(0, int(cz - pad)), min(nz, int(cz + pad) + 1)
        y0, y1 = max(0, int(cy - pad)), min(ny, int(cy + pad) + 1)
        x0, x1 = max(0, int(cx - pad)), min(nx, int(cx + pad) + 1)
        if z0 >= z1 or y0 >= y1 or x0 >= x1:
            continue
        d = np.sqrt((x[:, :, x0:x1] - cx) ** 2 + (y[:, y0:y1, :] - cy) ** 2 + (z[z0:z1, :, :] - cz) ** 2)
        val = 1e-4 + (1.0 - 1e-4) * 0.5 * (1.0 + np.tanh((d - R) / 1.0))
        sub = xhi[z0:z1, y0:y1, x0:x1]
        np.minimum(sub, val, out=sub)
    return xhi


def make_fields(name: str, dims=None, seed=None):
    """Return (kappa, S) as fp32 arrays [nbins][nz][ny][nx] for config `name` ("C1".."C5").

    `dims` overrides the mesh size (same generator, same seed) for reduced-size parity cases;
    `seed` overrides the config's seed (further realisations of the same recipe).
    """
    spec = CONFIGS[name]
    dims = tuple(dims) if dims is not None else spec.dims
    nx, ny, nz = dims
    rng = np.random.default_rng(spec.seed if seed is None else seed)
    if spec.kind == "uniform":
        kappa = rng.uniform(0.05, 2.0, size=(nz, ny, nx))
        S = rng.uniform(0.0, 1.0, size=(nz, ny, nx))
    else:
        g = _gaussian_field(rng, dims)
        n = np.exp(spec.sigma * g - 0.5 * spec.sigma * spec.sigma)
        del g
        c = 0.5 / np.median(n)                      # median dtau per cell = 0.5 at x_HI = 1
        n2mean = np.mean(n * n)
        if spec.kind == "lognormal":
            kappa = c * n
            S = n * n / n2mean
        else:
            xhi = _bubble_xhi(rng, dims, spec.nbubbles)
            kappa = c * n * xhi
            S = n * n * (1.0 - xhi) ** 2 / n2mean
            del xhi
        del n
        if spec.clip is not None:
            np.clip(kappa, spec.clip[0], spec.clip[1], out=kappa)
    ks, ss = [], []
    for nu in spec.nu:
        ks.append((kappa * nu ** -3.0).astype(np.float32))   # sigma_HI ~ nu^-3
        ss.append((S * nu ** 4.0).astype(np.float32))        # S_nu ~ h nu / sigma_HI(nu)  (eq. 18 shape)
    return np.stack(ks), np.stack(ss)
