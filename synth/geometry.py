"""Synthetic UT geometry table (stands in for the LHCb conditions).

BASELINE.json configs[0]: 4 layers at z = 2327.5, 2372.5, 2597.5, 2642.5 mm with
stereo slopes dxdy = 0, +tan5deg, -tan5deg, 0 (UTaX, UTaU, UTbV, UTbX,
PAPER.md:151); each layer 16 columns x 14 rows of 96 x 96 mm sectors covering
x in [-768, 768], y in [-672, 672]; 512 strips of 0.1875 mm per sector.

A *sector group* (hits "guaranteed to be within certain X
coordinates") is one column of 14 sectors in one layer: 16 per layer, 64 per
event.  Dense sector index s = layer*224 + col*14 + row, so a
group's sectors are contiguous; raw (on-the-wire) id = layer*256 + col*16 + row.

Everything here is table data (inputs to both implementations), computed in
float64 and rounded to float32 exactly once.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

N_LAYERS = 4
N_COLS = 16
N_ROWS = 14
N_STRIPS = 512
PITCH = 0.1875            # mm
SECTOR_W = 96.0           # mm = 512 * 0.1875
SECTOR_H = 96.0
X_MIN = -768.0
Y_MIN = -672.0
HOLE_HALF = 48.0          # beam hole |x|,|y| < 48 mm
LAYER_Z = (2327.5, 2372.5, 2597.5, 2642.5)
TAN5 = math.tan(math.radians(5.0))
LAYER_DXDY = (0.0, TAN5, -TAN5, 0.0)
INVALID = 0xFFFFFFFF
GROUP_MARGIN = 1e-3       # mm, outward widening of group bounds (covers fp32 rounding of x)


@dataclass
class UTGeometry:
    n_layers: int
    n_sectors: int
    n_groups: int
    id_to_sector: np.ndarray      # u32 [id_table_size], INVALID where unused
    sector_raw_id: np.ndarray     # u32 [n_sectors]
    sector_group: np.ndarray      # u32 [n_sectors], non-decreasing
    group_first_sector: np.ndarray  # u32 [n_groups+1]
    x0: np.ndarray                # f32 [n_sectors]  x_left - dxdy*y_c
    pitch: np.ndarray
    dxdy: np.ndarray
    z: np.ndarray
    y_begin: np.ndarray
    y_end: np.ndarray
    weight: np.ndarray            # 12 / pitch^2
    group_xmin: np.ndarray        # f32 [n_groups]
    group_xmax: np.ndarray
    layer_z: np.ndarray           # f32 [4]
    layer_dxdy: np.ndarray        # f32 [4]
    # float64 helpers for the generator only
    x_left64: np.ndarray = field(repr=False, default=None)
    y_c64: np.ndarray = field(repr=False, default=None)
    # optional position-dependent kick table (synth/field.py), None = constant kick
    kick: object = field(repr=False, default=None)

    @property
    def id_table_size(self) -> int:
        return int(self.id_to_sector.shape[0])

    @property
    def groups_per_layer(self) -> int:
        return self.n_groups // self.n_layers


def dense_sector(layer, col, row):
    return layer * (N_COLS * N_ROWS) + col * N_ROWS + row


def raw_sector_id(layer, col, row):
    return layer * 256 + col * 16 + row


def make_geometry() -> UTGeometry:
    n_sectors = N_LAYERS * N_COLS * N_ROWS
    n_groups = N_LAYERS * N_COLS
    layer = np.repeat(np.arange(N_LAYERS), N_COLS * N_ROWS)
    col = np.tile(np.repeat(np.arange(N_COLS), N_ROWS), N_LAYERS)
    row = np.tile(np.arange(N_ROWS), N_LAYERS * N_COLS)
    assert np.array_equal(dense_sector(layer, col, row), np.arange(n_sectors))

    raw_id = raw_sector_id(layer, col, row).astype(np.uint32)
    id_to_sector = np.full(1024, INVALID, dtype=np.uint32)
    id_to_sector[raw_id] = np.arange(n_sectors, dtype=np.uint32)

    dxdy64 = np.asarray(LAYER_DXDY, dtype=np.float64)[layer]
    z64 = np.asarray(LAYER_Z, dtype=np.float64)[layer]
    x_left = X_MIN + SECTOR_W * col
    y_lo = Y_MIN + SECTOR_H * row
    y_c = y_lo + 0.5 * SECTOR_H
    x0 = x_left - dxdy64 * y_c
    pitch = np.full(n_sectors, PITCH)
    weight = 12.0 / (pitch * pitch)

    group = (layer * N_COLS + col).astype(np.uint32)
    first = np.searchsorted(group, np.arange(n_groups + 1)).astype(np.uint32)
    # bounds of xAtYEq0 inside a group: strip centres span
    # [x0 + 0.25*pitch, x0 + (511 + 0.75)*pitch] for every row of the column
    lo = x0 + 0.25 * pitch
    hi = x0 + (N_STRIPS - 1 + 0.75) * pitch
    gmin = np.array([lo[group == g].min() for g in range(n_groups)]) - GROUP_MARGIN
    gmax = np.array([hi[group == g].max() for g in range(n_groups)]) + GROUP_MARGIN

    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return UTGeometry(
        n_layers=N_LAYERS, n_sectors=n_sectors, n_groups=n_groups,
        id_to_sector=id_to_sector, sector_raw_id=raw_id, sector_group=group,
        group_first_sector=first,
        x0=f32(x0), pitch=f32(pitch), dxdy=f32(dxdy64), z=f32(z64),
        y_begin=f32(y_lo), y_end=f32(y_lo + SECTOR_H), weight=f32(weight),
        group_xmin=f32(gmin), group_xmax=f32(gmax),
        layer_z=f32(LAYER_Z), layer_dxdy=f32(LAYER_DXDY),
        x_left64=x_left.astype(np.float64), y_c64=y_c.astype(np.float64),
    )
