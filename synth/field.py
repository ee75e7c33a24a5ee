"""Synthetic magnet look-up table (stands in for the LHCb field tables of: "look-up tables are used,
which give quick access to the influence of the magnetic field").

The constant kick of the base workloads (kappa = 60 MeV at z_mag = 1750 mm) becomes position dependent: the
integrated field falls off towards the edge of the magnet aperture and the effective kick plane moves with |y|.
A track looks its (kappa, z_mag) up ONCE, in the bin that holds its straight-line position at z_ref (nearest bin,
no interpolation, so that both implementations index the same cell):

    x_k = x_v + tx * (z_ref - z_v),  y_k = y_v + ty * (z_ref - z_v)                    (fp32, written order)
    ix = clamp(floor((x_k - x_lo) * inv_dx), 0, nx - 1),  iy likewise  (NaN -> 0);   cell = iy * nx + ix

Table data only (float64 -> float32 once); the generator bends its tracks with the same table.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class KickLUT:
    nx: int
    ny: int
    x_lo: float
    y_lo: float
    inv_dx: float
    inv_dy: float
    z_ref: float
    kappa: np.ndarray      # f32 [ny * nx]  MeV
    z_mag: np.ndarray      # f32 [ny * nx]  mm

    def cell64(self, x, y):
        """float64 bin index of positions (generator side)."""
        ix = np.clip(np.floor((np.asarray(x, np.float64) - self.x_lo) * self.inv_dx), 0, self.nx - 1).astype(np.int64)
        iy = np.clip(np.floor((np.asarray(y, np.float64) - self.y_lo) * self.inv_dy), 0, self.ny - 1).astype(np.int64)
        return iy * self.nx + ix


def make_kick_lut(nx: int = 24, ny: int = 20, half_x: float = 600.0, half_y: float = 500.0, z_ref: float = 1750.0,
                  kappa0: float = 60.0, z_mag0: float = 1750.0, falloff: float = 0.12, bow: float = 40.0) -> KickLUT:
    f = lambda v: float(np.float32(v))
    dx, dy = 2.0 * half_x / nx, 2.0 * half_y / ny
    xc = -half_x + dx * (np.arange(nx) + 0.5)
    yc = -half_y + dy * (np.arange(ny) + 0.5)
    X, Y = np.meshgrid(xc, yc)                                   # [ny, nx]
    r2 = (X / half_x) ** 2 + (Y / half_y) ** 2
    kappa = kappa0 * (1.0 - falloff * np.minimum(r2, 2.0) / 2.0)  # weaker integrated field towards the aperture edge
    z_mag = z_mag0 + bow * (Y / half_y) ** 2 - 0.5 * bow * (X / half_x) ** 2
    return KickLUT(nx, ny, f(-half_x), f(-half_y), f(1.0 / dx), f(1.0 / dy), f(z_ref),
                   np.ascontiguousarray(kappa.ravel(), np.float32), np.ascontiguousarray(z_mag.ravel(), np.float32))
