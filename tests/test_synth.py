"""Generator and raw-format checks (no method arithmetic is exercised here)."""
import struct

import numpy as np
import pytest

import synth
from synth import geometry as G
from synth.events import EventModel, encode_event, generate_event, generate_batch


def parse_raw(raw: bytes, offs, geom):
    """Independent pure-Python reader of the synthetic bank format (PAPER.md:239 stand-in)."""
    out = []
    for j in range(len(offs) - 1):
        o0, o1 = int(offs[j]), int(offs[j + 1])
        rid, cnt = struct.unpack_from("<IH", raw, o0)
        assert o1 - o0 == (6 + 2 * cnt + 3) // 4 * 4
        assert o0 % 4 == 0
        words = struct.unpack_from(f"<{cnt}H", raw, o0 + 6)
        pad = raw[o0 + 6 + 2 * cnt:o1]
        assert all(b == 0 for b in pad)
        s = int(geom.id_to_sector[rid])
        assert s != G.INVALID
        out.append((s, [(w & 0x1FF, (w >> 9) & 1, w >> 10) for w in words]))
    return out


@pytest.mark.parametrize("shuffle", [False, True])
def test_encode_round_trip(geom, shuffle):
    rng = np.random.default_rng(7)
    n = 3000
    sector = rng.integers(0, geom.n_sectors, n)
    strip = rng.integers(0, 512, n)
    frac = rng.integers(0, 2, n)
    adc = rng.integers(0, 64, n)
    order = rng.permutation(geom.n_sectors) if shuffle else None
    raw, offs = encode_event(geom, sector, strip, frac, adc, order)
    banks = parse_raw(raw.tobytes(), offs, geom)
    assert len(banks) == geom.n_sectors
    assert sorted(b[0] for b in banks) == list(range(geom.n_sectors))
    got = sorted((s, st, fr, a) for s, ws in banks for (st, fr, a) in ws)
    want = sorted(zip(sector.tolist(), strip.tolist(), frac.tolist(), adc.tolist()))
    assert got == want
    # emission order survives inside a bank
    for s, ws in banks:
        sel = np.nonzero(sector == s)[0]
        assert [w[0] for w in ws] == strip[sel].tolist()
    if shuffle:
        assert [b[0] for b in banks] == order.tolist()


def test_geometry_tables(geom):
    assert geom.n_sectors == 896 and geom.n_groups == 64 and geom.n_layers == 4
    assert np.all(np.diff(geom.sector_group.astype(np.int64)) >= 0)
    assert np.array_equal(geom.id_to_sector[geom.sector_raw_id], np.arange(896))
    assert (geom.id_to_sector != G.INVALID).sum() == 896
    assert np.allclose(geom.weight, 12.0 / 0.1875 ** 2)
    # group bounds non-decreasing inside a layer (contract used by the window lookup)
    for l in range(4):
        sl = slice(16 * l, 16 * l + 16)
        assert np.all(np.diff(geom.group_xmin[sl]) > 0) and np.all(np.diff(geom.group_xmax[sl]) > 0)
    # stereo groups are widened by |dxdy| * 624 mm and overlap their neighbours
    assert geom.group_xmax[16] - geom.group_xmin[16] == pytest.approx(96 + 2 * 624 * G.TAN5, abs=0.5)
    assert geom.group_xmax[0] - geom.group_xmin[0] == pytest.approx(96, abs=0.5)


def test_event_independent_of_batch(geom):
    m = EventModel()
    b = generate_batch(geom, m, seed=11, n_events=4)
    e2 = generate_event(geom, m, 11, 2)
    ns = geom.n_sectors
    lo, hi = int(b.bank_offsets[2 * ns]), int(b.bank_offsets[3 * ns])
    assert np.array_equal(b.raw[lo:hi], e2["raw"])
    v0, v1 = int(b.velo_offsets[2]), int(b.velo_offsets[3])
    assert np.array_equal(b.velo_x[v0:v1], e2["velo"][0])
    b2 = generate_batch(geom, m, seed=11, n_events=2, first_event=2)
    assert np.array_equal(b2.raw[:hi - lo], e2["raw"])


def test_config_shapes(wl):
    geom, b, p = wl(2)
    assert b.n_events == 100
    assert 1850 < b.total_hits / 100 < 2150            # "~2000 UT hits" per event
    assert 140 < b.n_velo_total / 100 < 160            # Poisson(150)
    assert b.bank_offsets.shape[0] == 100 * 896 + 1
    assert b.hit_capacity >= b.total_hits
    assert p.min_hits == 3 and p.max_candidates_per_layer == 16
    # win_half = (kappa/p_min) * (z - z_mag) + 0.5
    assert p.win_half[0] == pytest.approx(60 / 2000 * (2327.5 - 1750) + 0.5, rel=1e-6)
    geom, b1, p1 = wl(1)
    assert b1.n_events == 1 and b1.n_velo_total == 20 and 40 <= b1.total_hits <= 80


def test_unique_strip_per_sector(geom):
    e = generate_event(geom, EventModel(mean_tracks=600, noise_mean=6000), 4, 0)
    banks = parse_raw(e["raw"].tobytes(), e["bank_offs"], geom)
    for s, ws in banks:
        strips = [w[0] for w in ws]
        assert len(strips) == len(set(strips))
    assert sum(len(ws) for _, ws in banks) == e["n_hits"]
