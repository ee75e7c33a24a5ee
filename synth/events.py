"""Seeded synthetic collision events: VELO states, UT raw banks and generator truth.

Recipe: SURVEY.md section 8(d) / BASELINE.json configs[0..1].  Stands in for the
LHCb minbias / Bs->phiphi Monte-Carlo of PAPER.md:364-368 (not available here).

Raw-bank format (synthetic stand-in for the "highly compact format" of
PAPER.md:239): one bank per sector and event, 4-byte aligned,
    u32 raw sector id | u16 count | count x u16 word | zero pad to 4 bytes
    word = 9-bit strip | frac << 9 | 6-bit ADC << 10
Banks of one event are contiguous, in any order; ``bank_offsets`` holds the
byte offset of every bank plus the end (n_events * n_sectors + 1 entries).

This module ENcodes; it never decodes.  Every random number comes from
``numpy.random.default_rng([seed, event])`` so an event does not depend on
the batch it is generated in.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

from . import geometry as G

Z_VELO = 770.0      # mm, z of the VELO state
Z_MAG = 1750.0      # mm, kick plane
KAPPA = 60.0        # MeV, integrated-field kick: dx/dz changes by KAPPA * q / p


@dataclass(frozen=True)
class EventModel:
    """Per-event generator parameters (BASELINE.json configs)."""
    mean_tracks: float = 150.0        # Poisson mean; ignored when fixed_tracks >= 0
    fixed_tracks: int = -1
    efficiency: float = 0.97
    noise_mean: float = 1500.0        # Poisson mean of noise words per event
    sigma_hit: float = 0.05           # mm
    p_min_gev: float = 2.0
    p_max_gev: float = 100.0
    shuffle_banks: bool = True        # banks of an event in random order


@dataclass
class Batch:
    """A batch of events as the two ABI calls consume it, plus truth."""
    n_events: int
    raw: np.ndarray            # u8 [total_bytes]
    bank_offsets: np.ndarray   # u32 [n_events*n_sectors + 1]
    velo_x: np.ndarray         # f32 [n_velo_total]
    velo_y: np.ndarray
    velo_tx: np.ndarray
    velo_ty: np.ndarray
    velo_offsets: np.ndarray   # u32 [n_events + 1]
    velo_z: float
    # truth (never seen by the algorithms)
    truth_hit_id: np.ndarray   # i64 [n_velo_total, 4]: id of the recorded hit of track t in layer l, or -1
    truth_q: np.ndarray        # i8  [n_velo_total]
    truth_p: np.ndarray        # f64 [n_velo_total] MeV
    n_hits_event: np.ndarray   # i64 [n_events] words actually encoded
    hit_capacity: int = 0      # (total_raw_bytes - 6*n_banks)//2: upper bound known from sizes alone

    @property
    def n_velo_total(self) -> int:
        return int(self.velo_offsets[-1])

    @property
    def total_hits(self) -> int:
        return int(self.n_hits_event.sum())


def encode_event(geom: G.UTGeometry, sector: np.ndarray, strip: np.ndarray, frac: np.ndarray,
                 adc: np.ndarray, bank_order: np.ndarray | None = None):
    """Pack hits (dense sector, strip, frac, adc), given in emission order, into the
    raw banks of one event.  Returns (raw_u8, bank_byte_offsets[n_sectors+1])."""
    ns = geom.n_sectors
    sector = np.asarray(sector, dtype=np.int64)
    if bank_order is None:
        bank_order = np.arange(ns)
    bank_pos = np.empty(ns, dtype=np.int64)          # sector -> position in the event's bank sequence
    bank_pos[bank_order] = np.arange(ns)
    counts = np.bincount(sector, minlength=ns)[bank_order]   # per bank position
    if counts.max(initial=0) > 0xFFFF:
        raise ValueError("bank count does not fit u16")
    size = 6 + 2 * counts
    size = (size + 3) & ~3
    offs = np.zeros(ns + 1, dtype=np.int64)
    np.cumsum(size, out=offs[1:])
    raw16 = np.zeros(offs[-1] // 2, dtype=np.uint16)
    ids = geom.sector_raw_id[bank_order].astype(np.uint32)
    h = offs[:-1] // 2
    raw16[h] = (ids & 0xFFFF).astype(np.uint16)
    raw16[h + 1] = (ids >> 16).astype(np.uint16)
    raw16[h + 2] = counts.astype(np.uint16)
    if sector.size:
        pos = bank_pos[sector]
        order = np.argsort(pos, kind="stable")        # emission order survives inside a bank
        pos_s = pos[order]
        start = np.zeros(ns, dtype=np.int64)
        np.cumsum(counts[:-1], out=start[1:])
        k = np.arange(sector.size) - start[pos_s]
        word = (np.asarray(strip, dtype=np.int64) & 0x1FF) | ((np.asarray(frac, dtype=np.int64) & 1) << 9) \
            | ((np.asarray(adc, dtype=np.int64) & 0x3F) << 10)
        raw16[h[pos_s] + 3 + k] = word[order].astype(np.uint16)
    return raw16.view(np.uint8), offs


def generate_event(geom: G.UTGeometry, model: EventModel, seed: int, event: int):
    """One event.  Returns dict(raw, bank_offs, velo[4 arrays], truth_hit_id, q, p, n_hits)."""
    rng = np.random.default_rng([seed, event])
    T = model.fixed_tracks if model.fixed_tracks >= 0 else int(rng.poisson(model.mean_tracks))
    ox = rng.normal(0.0, 0.05, T)
    oy = rng.normal(0.0, 0.05, T)
    oz = rng.normal(0.0, 50.0, T)
    eta = rng.uniform(2.0, 5.0, T)
    phi = rng.uniform(0.0, 2.0 * math.pi, T)
    q = (rng.integers(0, 2, T) * 2 - 1).astype(np.int8)
    p = np.exp(rng.uniform(math.log(model.p_min_gev * 1e3), math.log(model.p_max_gev * 1e3), T))  # MeV
    theta = 2.0 * np.arctan(np.exp(-eta))
    tx = np.tan(theta) * np.cos(phi)
    ty = np.tan(theta) * np.sin(phi)
    xv = ox + tx * (Z_VELO - oz)
    yv = oy + ty * (Z_VELO - oz)

    zl = np.asarray(G.LAYER_Z)[None, :]
    dxdy = np.asarray(G.LAYER_DXDY)[None, :]
    kap, zm = np.full(T, KAPPA), np.full(T, Z_MAG)
    if geom.kick is not None:                              # position-dependent kick (synth/field.py)
        lut = geom.kick
        cell = lut.cell64(xv + tx * (lut.z_ref - Z_VELO), yv + ty * (lut.z_ref - Z_VELO))
        kap, zm = lut.kappa[cell].astype(np.float64), lut.z_mag[cell].astype(np.float64)
    x = xv[:, None] + tx[:, None] * (zl - Z_VELO) + (kap * q / p)[:, None] * (zl - zm[:, None])
    y = yv[:, None] + ty[:, None] * (zl - Z_VELO)
    smear = rng.normal(0.0, model.sigma_hit, (T, 4))
    keep_draw = rng.uniform(0.0, 1.0, (T, 4))
    adc_true = rng.integers(0, 64, (T, 4))
    acc = (np.abs(x) < -G.X_MIN) & (np.abs(y) < -G.Y_MIN) & ~((np.abs(x) < G.HOLE_HALF) & (np.abs(y) < G.HOLE_HALF))
    row = np.clip(np.floor((y - G.Y_MIN) / G.SECTOR_H).astype(np.int64), 0, G.N_ROWS - 1)
    y_c = G.Y_MIN + G.SECTOR_H * row + 0.5 * G.SECTOR_H
    xs = x - dxdy * (y - y_c) + smear                      # column from xs
    col = np.floor((xs - G.X_MIN) / G.SECTOR_W).astype(np.int64)
    ok = acc & (col >= 0) & (col < G.N_COLS) & (keep_draw < model.efficiency)
    colc = np.clip(col, 0, G.N_COLS - 1)
    local = (xs - (G.X_MIN + G.SECTOR_W * colc)) / G.PITCH
    strip = np.clip(np.floor(local).astype(np.int64), 0, G.N_STRIPS - 1)
    frac = ((local - strip) >= 0.5).astype(np.int64)
    layer = np.broadcast_to(np.arange(4)[None, :], (T, 4))
    sec_true = G.dense_sector(layer, colc, row)

    n_noise = int(rng.poisson(model.noise_mean)) if model.noise_mean > 0 else 0
    sec_n = rng.integers(0, geom.n_sectors, n_noise)
    strip_n = rng.integers(0, G.N_STRIPS, n_noise)
    frac_n = rng.integers(0, 2, n_noise)
    adc_n = rng.integers(0, 64, n_noise)

    sel = np.nonzero(ok.ravel())[0]                      # track-major, layer-minor emission order
    sector = np.concatenate([sec_true.ravel()[sel], sec_n])
    strips = np.concatenate([strip.ravel()[sel], strip_n])
    fracs = np.concatenate([frac.ravel()[sel], frac_n])
    adcs = np.concatenate([adc_true.ravel()[sel], adc_n])
    owner = np.concatenate([sel, np.full(n_noise, -1, dtype=np.int64)])   # flat (track*4+layer) or -1

    # one word per (sector, strip); first writer wins (true hits precede noise)
    key = sector * G.N_STRIPS + strips
    _, first = np.unique(key, return_index=True)
    first.sort()
    sector, strips, fracs, adcs, owner = sector[first], strips[first], fracs[first], adcs[first], owner[first]

    bank_order = rng.permutation(geom.n_sectors) if model.shuffle_banks else None
    raw, offs = encode_event(geom, sector, strips, fracs, adcs, bank_order)

    truth = np.full(T * 4, -1, dtype=np.int64)
    own = owner >= 0
    hit_id = (geom.sector_raw_id[sector].astype(np.int64) << 9) | strips
    truth[owner[own]] = hit_id[own]
    return dict(raw=raw, bank_offs=offs,
                velo=(xv.astype(np.float32), yv.astype(np.float32), tx.astype(np.float32), ty.astype(np.float32)),
                truth_hit_id=truth.reshape(T, 4), q=q, p=p, n_hits=int(sector.size))


def assemble_batch(geom: G.UTGeometry, events: list) -> Batch:
    n_events = len(events)
    ns = geom.n_sectors
    sizes = np.array([e["raw"].size for e in events], dtype=np.int64)
    base = np.zeros(n_events + 1, dtype=np.int64)
    np.cumsum(sizes, out=base[1:])
    if base[-1] >= 2 ** 32:
        raise ValueError("raw batch exceeds u32 byte offsets")
    bank_offsets = np.empty(n_events * ns + 1, dtype=np.uint32)
    for i, e in enumerate(events):
        bank_offsets[i * ns:(i + 1) * ns] = (e["bank_offs"][:-1] + base[i]).astype(np.uint32)
    bank_offsets[-1] = base[-1]
    raw = np.concatenate([e["raw"] for e in events]) if n_events else np.zeros(0, np.uint8)
    nv = np.array([e["velo"][0].size for e in events], dtype=np.int64)
    velo_offsets = np.zeros(n_events + 1, dtype=np.uint32)
    velo_offsets[1:] = np.cumsum(nv)
    cat = lambda j: (np.concatenate([e["velo"][j] for e in events]).astype(np.float32)
                     if n_events else np.zeros(0, np.float32))
    empty = lambda dt, shape=(0,): np.zeros(shape, dt)
    return Batch(
        n_events=n_events, raw=np.ascontiguousarray(raw), bank_offsets=bank_offsets,
        velo_x=cat(0), velo_y=cat(1), velo_tx=cat(2), velo_ty=cat(3),
        velo_offsets=velo_offsets, velo_z=Z_VELO,
        truth_hit_id=np.concatenate([e["truth_hit_id"] for e in events]) if n_events else empty(np.int64, (0, 4)),
        truth_q=np.concatenate([e["q"] for e in events]) if n_events else empty(np.int8),
        truth_p=np.concatenate([e["p"] for e in events]) if n_events else empty(np.float64),
        n_hits_event=np.array([e["n_hits"] for e in events], dtype=np.int64),
        hit_capacity=int((base[-1] - 6 * n_events * ns) // 2),
    )


def _gen_range(args):
    model, seed, lo, hi, kick = args
    geom = G.make_geometry()
    geom.kick = kick
    return [generate_event(geom, model, seed, ev) for ev in range(lo, hi)]


def generate_batch(geom: G.UTGeometry, model: EventModel, seed: int, n_events: int,
                   first_event: int = 0, workers: int = 1) -> Batch:
    """Events first_event .. first_event+n_events-1 of stream ``seed``."""
    if workers > 1 and n_events >= 4 * workers:
        import multiprocessing as mp
        cuts = np.linspace(first_event, first_event + n_events, workers + 1).astype(int)
        with mp.get_context("fork").Pool(workers) as pool:
            parts = pool.map(_gen_range, [(model, seed, int(a), int(b), geom.kick) for a, b in zip(cuts[:-1], cuts[1:])])
        events = [e for part in parts for e in part]
    else:
        events = [generate_event(geom, model, seed, ev) for ev in range(first_event, first_event + n_events)]
    return assemble_batch(geom, events)
