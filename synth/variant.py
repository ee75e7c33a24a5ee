"""A second, non-uniform synthetic UT geometry and a table-driven event generator for it.

SURVEY.md 8(f) row 3 asks for a UT-like layout "with finer inner sectors, staves and overlaps"
(sector groups are "narrower at the centre").  Both implementations are driven by
the geometry TABLES, so this layout exists to catch any hidden dependence on the regular 16 x 14 layout
of ``geometry.make_geometry``:

* 14 columns per layer: 5 outer (96 mm, pitch 0.1875), 4 inner (48 mm, pitch 0.09375), 5 outer;
* 16 rows per column: 6 tall (96 mm), 4 short (48 mm) around y = 0, 6 tall; neighbouring rows
  OVERLAP by 2 mm in y (a track near a boundary crosses two sectors of one group);
* z staggered per sector by +-5 mm around the layer z (front / back of a stave), so a hit's z is not the
  layer's z;
* raw ids spread over a 4096-entry table (layer*1024 + col*64 + row*3 + 1);
* optionally the rows of every column stored in a shuffled order (the "rows not sorted" path).

Group = column (56 groups of 16 sectors).  Input generation only -- no decoding, no search, no fit.
"""
from __future__ import annotations

import math

import numpy as np

from . import geometry as G
from .events import EventModel, Batch, encode_event, assemble_batch, Z_VELO, Z_MAG, KAPPA

COL_W = (96.0,) * 5 + (48.0,) * 4 + (96.0,) * 5
ROW_H = (96.0,) * 6 + (48.0,) * 4 + (96.0,) * 6
Y_OVERLAP = 1.0           # every sector is extended by this much at both ends
Z_STAGGER = 5.0


def make_staggered_geometry(shuffle_rows: bool = False, seed: int = 7) -> G.UTGeometry:
    nc, nr = len(COL_W), len(ROW_H)
    n_sectors, n_groups = G.N_LAYERS * nc * nr, G.N_LAYERS * nc
    x_edges = np.concatenate([[0.0], np.cumsum(COL_W)]) - 0.5 * sum(COL_W)
    y_edges = np.concatenate([[0.0], np.cumsum(ROW_H)]) - 0.5 * sum(ROW_H)
    rng = np.random.default_rng(seed)
    layer = np.repeat(np.arange(G.N_LAYERS), nc * nr)
    col = np.tile(np.repeat(np.arange(nc), nr), G.N_LAYERS)
    row = np.tile(np.arange(nr), G.N_LAYERS * nc)
    if shuffle_rows:                                    # dense order inside a column is no longer y order
        row = np.concatenate([rng.permutation(nr) for _ in range(G.N_LAYERS * nc)])
    raw_id = (layer * 1024 + col * 64 + row * 3 + 1).astype(np.uint32)
    id_to_sector = np.full(4096, G.INVALID, dtype=np.uint32)
    id_to_sector[raw_id] = np.arange(n_sectors, dtype=np.uint32)

    dxdy64 = np.asarray(G.LAYER_DXDY, dtype=np.float64)[layer]
    z64 = np.asarray(G.LAYER_Z, dtype=np.float64)[layer] + Z_STAGGER * np.where((col + row) % 2 == 0, 1.0, -1.0)
    x_left = x_edges[col]
    pitch = np.asarray(COL_W)[col] / G.N_STRIPS
    y_lo, y_hi = y_edges[row] - Y_OVERLAP, y_edges[row + 1] + Y_OVERLAP
    y_c = 0.5 * (y_lo + y_hi)
    x0 = x_left - dxdy64 * y_c
    group = (layer * nc + col).astype(np.uint32)
    first = np.searchsorted(group, np.arange(n_groups + 1)).astype(np.uint32)
    lo = x0 + 0.25 * pitch
    hi = x0 + (G.N_STRIPS - 1 + 0.75) * pitch
    gmin = np.array([lo[group == g].min() for g in range(n_groups)]) - G.GROUP_MARGIN
    gmax = np.array([hi[group == g].max() for g in range(n_groups)]) + G.GROUP_MARGIN
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return G.UTGeometry(
        n_layers=G.N_LAYERS, n_sectors=n_sectors, n_groups=n_groups, id_to_sector=id_to_sector,
        sector_raw_id=raw_id, sector_group=group, group_first_sector=first,
        x0=f32(x0), pitch=f32(pitch), dxdy=f32(dxdy64), z=f32(z64), y_begin=f32(y_lo), y_end=f32(y_hi),
        weight=f32(12.0 / (pitch * pitch)), group_xmin=f32(gmin), group_xmax=f32(gmax),
        layer_z=f32(G.LAYER_Z), layer_dxdy=f32(G.LAYER_DXDY),
        x_left64=x_left.astype(np.float64), y_c64=y_c.astype(np.float64))


def generate_event_tables(geom: G.UTGeometry, model: EventModel, seed: int, event: int):
    """One event on ANY geometry table: a track leaves a hit in every sector of a layer whose y range and
    strip range contain it (overlapping rows give two hits).  Same kinematics as events.generate_event."""
    rng = np.random.default_rng([seed, event, 1])
    T = model.fixed_tracks if model.fixed_tracks >= 0 else int(rng.poisson(model.mean_tracks))
    ox, oy, oz = rng.normal(0.0, 0.05, T), rng.normal(0.0, 0.05, T), rng.normal(0.0, 50.0, T)
    eta, phi = rng.uniform(2.0, 5.0, T), rng.uniform(0.0, 2.0 * math.pi, T)
    q = (rng.integers(0, 2, T) * 2 - 1).astype(np.int8)
    p = np.exp(rng.uniform(math.log(model.p_min_gev * 1e3), math.log(model.p_max_gev * 1e3), T))
    theta = 2.0 * np.arctan(np.exp(-eta))
    tx, ty = np.tan(theta) * np.cos(phi), np.tan(theta) * np.sin(phi)
    xv, yv = ox + tx * (Z_VELO - oz), oy + ty * (Z_VELO - oz)

    x0 = geom.x0.astype(np.float64); pitch = geom.pitch.astype(np.float64); sl = geom.dxdy.astype(np.float64)
    zs = geom.z.astype(np.float64); yb = geom.y_begin.astype(np.float64); ye = geom.y_end.astype(np.float64)
    spl = geom.n_sectors // geom.n_layers
    sec, strip, frac = [], [], []
    for l in range(geom.n_layers):
        s = np.arange(l * spl, (l + 1) * spl)
        z = zs[s][None, :]                                           # the sector's own (staggered) z
        x = xv[:, None] + tx[:, None] * (z - Z_VELO) + KAPPA * (q / p)[:, None] * (z - Z_MAG)
        y = yv[:, None] + ty[:, None] * (z - Z_VELO)
        xs = x - sl[s][None, :] * y + rng.normal(0.0, model.sigma_hit, (T, 1))
        u = (xs - x0[s][None, :]) / pitch[s][None, :]
        ok = (y >= yb[s][None, :]) & (y <= ye[s][None, :]) & (u >= 0) & (u < G.N_STRIPS)
        ok &= ~((np.abs(x) < G.HOLE_HALF) & (np.abs(y) < G.HOLE_HALF))
        ok &= rng.random((T, 1)) < model.efficiency
        ti, si = np.nonzero(ok)
        st = np.floor(u[ti, si]).astype(np.int64)
        sec.append(s[si]); strip.append(st); frac.append(((u[ti, si] - st) >= 0.5).astype(np.int64))
    n_noise = int(rng.poisson(model.noise_mean))
    sec.append(rng.integers(0, geom.n_sectors, n_noise)); strip.append(rng.integers(0, G.N_STRIPS, n_noise))
    frac.append(rng.integers(0, 2, n_noise))
    sec, strip, frac = np.concatenate(sec), np.concatenate(strip), np.concatenate(frac)
    _, keep = np.unique(sec * G.N_STRIPS + strip, return_index=True)  # one word per (sector, strip): first writer wins
    keep.sort()
    sec, strip, frac = sec[keep], strip[keep], frac[keep]
    order = rng.permutation(geom.n_sectors) if model.shuffle_banks else None
    raw, offs = encode_event(geom, sec, strip, frac, rng.integers(0, 64, sec.size), order)
    f32 = lambda a: a.astype(np.float32)
    return dict(raw=raw, bank_offs=offs, velo=(f32(xv), f32(yv), f32(tx), f32(ty)),
                truth_hit_id=np.full((T, 4), -1, np.int64), q=q, p=p, n_hits=int(sec.size))


def generate_batch_tables(geom: G.UTGeometry, model: EventModel, seed: int, n_events: int) -> Batch:
    return assemble_batch(geom, [generate_event_tables(geom, model, seed, ev) for ev in range(n_events)])
