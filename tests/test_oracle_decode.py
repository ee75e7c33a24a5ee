"""Pins of the decode oracle: none of them re-calls the oracle's own
formula in fp32 -- they use float64 closed forms, invariants, round trips and hand-built banks."""
import numpy as np
import pytest

import oracle
import synth
from synth import geometry as G
from synth.events import encode_event, KAPPA, Z_MAG, Z_VELO


def one_event(geom, sector, strip, frac, order=None):
    n = len(sector)
    raw, offs = encode_event(geom, np.asarray(sector), np.asarray(strip), np.asarray(frac), np.zeros(n, int), order)
    return raw, offs.astype(np.uint32)


def x_expected64(geom, s, strip, frac):
    """float64 closed form of SURVEY.md A3: x_left - dxdy*y_c + (strip + 0.25 + 0.5 frac) * pitch."""
    layer = s // 224
    return geom.x_left64[s] - np.asarray(G.LAYER_DXDY)[layer] * geom.y_c64[s] + (strip + 0.25 + 0.5 * frac) * G.PITCH


def test_round_trip_ids_and_x(geom):
    rng = np.random.default_rng(3)
    key = rng.choice(896 * 512, 5000, replace=False)
    sector, strip = key // 512, key % 512
    frac = rng.integers(0, 2, 5000)
    raw, offs = one_event(geom, sector, strip, frac, rng.permutation(896))
    h = oracle.decode(raw, offs, 1, geom)
    assert h.status == 0 and h.n_hits == 5000
    want_id = (geom.sector_raw_id[sector].astype(np.int64) << 9) | strip
    assert sorted(h.id[:5000].tolist()) == sorted(want_id.tolist())        # ids: a permutation of the input
    # every field of every hit, matched through the id
    pos = {int(i): k for k, i in enumerate(h.id[:5000])}
    k = np.array([pos[int(i)] for i in want_id])
    x64 = x_expected64(geom, sector, strip, frac)
    # three roundings: the x0 table entry, the product, the sum -> half an ulp each
    sp = lambda v: np.spacing(np.abs(v).astype(np.float32)).astype(np.float64)
    tol = 0.5 * (sp(x64) + sp(geom.x0[sector].astype(np.float64)) + sp(np.full(5000, 96.0)))
    assert np.all(np.abs(h.x_at_y0[k] - x64) <= tol)
    assert np.array_equal(h.z_at_y0[k], geom.z[sector])
    assert np.array_equal(h.y_begin[k], geom.y_begin[sector])
    assert np.array_equal(h.y_end[k], geom.y_end[sector])
    assert np.array_equal(h.dxdy[k], geom.dxdy[sector])
    assert np.array_equal(h.weight[k], geom.weight[sector])
    # frac is recoverable from x: half-strip bin centre
    bin64 = (h.x_at_y0[k].astype(np.float64) - (x64 - (strip + 0.25 + 0.5 * frac) * G.PITCH)) / G.PITCH
    assert np.array_equal(np.round((bin64 - 0.25) * 2).astype(int), 2 * strip + frac)


def test_x_layers_closed_form_one_ulp(geom):
    # X layers (dxdy = 0): x = x_left + (strip + 0.25 + 0.5 frac) * pitch, all exactly representable inputs
    sector = np.repeat(np.arange(0, 224, 7), 16)
    strip = np.tile(np.arange(0, 512, 32), 32)
    frac = (strip // 32) % 2
    raw, offs = one_event(geom, sector, strip, frac)
    h = oracle.decode(raw, offs, 1, geom)
    pos = {int(i): k for k, i in enumerate(h.id[:h.n_hits])}
    ids = (geom.sector_raw_id[sector].astype(np.int64) << 9) | strip
    k = np.array([pos[int(i)] for i in ids])
    x64 = geom.x_left64[sector] + (strip + 0.25 + 0.5 * frac) * G.PITCH
    assert np.all(np.abs(h.x_at_y0[k].astype(np.float64) - x64) <= 0.5 * np.spacing(np.abs(x64).astype(np.float32)))


def check_container(geom, batch, h):
    ne, ng = batch.n_events, geom.n_groups
    off = h.hit_offsets.astype(np.int64)
    assert off[0] == 0 and off[-1] == h.n_hits == batch.total_hits
    assert np.all(np.diff(off) >= 0)
    # per event totals = words encoded; = sum over banks of (bank_bytes - 6 - pad)/2 read from the headers
    ev = off[::ng]
    assert np.array_equal(np.diff(ev), batch.n_hits_event)
    x = h.x_at_y0[:h.n_hits]
    grp = np.repeat(np.arange(ne * ng), np.diff(off))
    same = grp[1:] == grp[:-1]
    assert np.all(x[1:][same] >= x[:-1][same])                       # non-decreasing x per group
    g = grp % ng
    assert np.all(x >= geom.group_xmin[g]) and np.all(x <= geom.group_xmax[g])
    # hits sit in the group of their sector (id -> raw sector id -> dense sector -> group)
    s = geom.id_to_sector[h.id[:h.n_hits] >> 9]
    assert np.array_equal(geom.sector_group[s], g)
    assert np.array_equal(h.z_at_y0[:h.n_hits], geom.z[s])
    # ties keep fill order: ascending dense sector (X layers: same strip in different rows)
    tie = same & (x[1:] == x[:-1])
    assert np.all(s[1:][tie].astype(np.int64) > s[:-1][tie].astype(np.int64))
    return int(tie.sum())


def test_container_invariants_config2(wl):
    geom, b, p = wl(2)
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    assert h.status == 0
    n_ties = check_container(geom, b, h)
    assert n_ties > 0          # the stable-tie rule is actually exercised
    # header-only count: sum over banks of u16 count
    cnt = 0
    raw = b.raw
    for o in b.bank_offsets[:-1][:896 * 3].astype(np.int64):
        cnt += int(raw[o + 4]) | (int(raw[o + 5]) << 8)
    assert cnt == int(b.n_hits_event[:3].sum())


def test_container_invariants_config1_and_4(wl):
    for cfg, n in ((1, None), (4, 5)):
        geom, b, p = wl(cfg, n)
        h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
        assert h.status == 0
        check_container(geom, b, h)


def test_resolution_statistic(wl):
    """RMS(x_decoded(y_true) - x_true) = sqrt(0.05^2 + (pitch/2)^2/12) = 0.0569 mm."""
    geom, b, p = wl(2)
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    res = []
    off = h.hit_offsets.astype(np.int64)
    for e in range(b.n_events):
        lo, hi = off[e * 64], off[(e + 1) * 64]
        pos = {int(i): lo + k for k, i in enumerate(h.id[lo:hi])}
        for t in range(int(b.velo_offsets[e]), int(b.velo_offsets[e + 1])):
            for l in range(4):
                hid = int(b.truth_hit_id[t, l])
                if hid < 0:
                    continue
                k = pos[hid]
                z = G.LAYER_Z[l]
                xt = float(b.velo_x[t]) + float(b.velo_tx[t]) * (z - Z_VELO) + KAPPA * b.truth_q[t] / b.truth_p[t] * (z - Z_MAG)
                yt = float(b.velo_y[t]) + float(b.velo_ty[t]) * (z - Z_VELO)
                res.append(float(h.x_at_y0[k]) + float(h.dxdy[k]) * yt - xt)
    res = np.asarray(res)
    assert len(res) > 40000
    assert abs(res.mean()) < 2e-3
    assert np.sqrt((res ** 2).mean()) == pytest.approx(np.sqrt(0.05 ** 2 + (G.PITCH / 2) ** 2 / 12), rel=0.03)


def test_stable_ties_hand_built(geom):
    # X layer 0, column 3: same strip/frac in rows 13, 0, 5 -> equal x, output must be rows 0, 5, 13
    rows = [13, 0, 5]
    sector = [G.dense_sector(0, 3, r) for r in rows] + [G.dense_sector(0, 3, 2)]
    strip = [100, 100, 100, 99]
    frac = [1, 1, 1, 1]
    raw, offs = one_event(geom, sector, strip, frac, np.random.default_rng(0).permutation(896))
    h = oracle.decode(raw, offs, 1, geom)
    assert h.n_hits == 4
    got_rows = [(int(i) >> 9) & 0xF for i in h.id[:4]]
    assert got_rows == [2, 0, 5, 13]
    assert h.x_at_y0[1] == h.x_at_y0[2] == h.x_at_y0[3] > h.x_at_y0[0]
    assert np.array_equal(h.hit_offsets[:5], [0, 0, 0, 0, 4])


def test_edge_cases(geom):
    # empty event
    raw, offs = one_event(geom, [], [], [])
    h = oracle.decode(raw, offs, 1, geom)
    assert h.n_hits == 0 and h.status == 0 and not h.hit_offsets.any()
    # no events at all
    h = oracle.decode(np.zeros(0, np.uint8), np.zeros(1, np.uint32), 0, geom)
    assert h.n_hits == 0 and h.hit_offsets.tolist() == [0]
    # one full 512-word bank (all strips, descending emission order) next to empty banks
    s = G.dense_sector(2, 7, 6)
    strips = np.arange(511, -1, -1)
    raw, offs = one_event(geom, np.full(512, s), strips, strips % 2)
    h = oracle.decode(raw, offs, 1, geom)
    assert h.n_hits == 512 and np.array_equal(h.id[:512] & 0x1FF, np.arange(512))
    assert np.all(np.diff(h.x_at_y0[:512]) > 0)
    # all hits of an event in one group (14 sectors x 512 strips), two events, second empty
    sec = np.repeat(np.arange(14) + G.dense_sector(1, 0, 0), 512)
    st = np.tile(np.arange(512), 14)
    rng = np.random.default_rng(5)
    perm = rng.permutation(sec.size)
    r1, o1 = one_event(geom, sec[perm], st[perm], np.zeros(sec.size, int))
    r2, o2 = one_event(geom, [], [], [])
    raw = np.concatenate([r1, r2])
    offs = np.concatenate([o1[:-1], o2 + o1[-1]]).astype(np.uint32)
    h = oracle.decode(raw, offs, 2, geom)
    assert h.n_hits == 14 * 512 and h.status == 0
    assert h.hit_offsets[16] == 0 and h.hit_offsets[17] == 14 * 512 and np.all(h.hit_offsets[17:] == 14 * 512)
    assert np.all(np.diff(h.x_at_y0[:h.n_hits]) >= 0)


def test_error_status(geom):
    raw, offs = one_event(geom, [5, 5, 9], [1, 2, 3], [0, 0, 0])
    # unknown sector id
    bad = raw.copy()
    bad[int(offs[0]):int(offs[0]) + 4] = np.frombuffer(np.uint32(15).tobytes(), np.uint8)
    assert oracle.decode(bad, offs, 1, geom).status & oracle.ST_UNKNOWN_SECTOR
    bad = raw.copy()
    bad[int(offs[0]):int(offs[0]) + 4] = np.frombuffer(np.uint32(5000).tobytes(), np.uint8)
    assert oracle.decode(bad, offs, 1, geom).status & oracle.ST_UNKNOWN_SECTOR
    # duplicate sector: bank 0 claims the id of bank 1
    bad = raw.copy()
    bad[int(offs[0]):int(offs[0]) + 4] = raw[int(offs[1]):int(offs[1]) + 4]
    st = oracle.decode(bad, offs, 1, geom).status
    assert st & oracle.ST_DUPLICATE_SECTOR
    # count disagrees with the bank size
    bad = raw.copy()
    bad[int(offs[5]) + 4] = 7
    assert oracle.decode(bad, offs, 1, geom).status & oracle.ST_BAD_BANK_SIZE
    # capacity overflow: nothing written past capacity, offsets still exact
    h = oracle.decode(raw, offs, 1, geom, capacity=2)
    assert h.status & oracle.ST_CAPACITY and h.hit_offsets[-1] == 3
    assert oracle.decode(raw, offs, 1, geom).status == 0


def test_bank_alignment_and_range_rule(geom):
    """DESIGN.md A22: a bank off a 4-byte boundary, or outside its event's byte range, is ignored and flagged even
    when its size field is consistent.  Expected hits come from the encoder inputs (which banks survive)."""
    import malformed
    raw, offs, want, j = malformed.misaligned_tail(geom)
    h = oracle.decode(raw, offs, 1, geom)
    assert h.status == oracle.ST_BAD_BANK_SIZE
    assert sorted(h.id[:h.n_hits].astype(np.int64).tolist()) == want
    # the same bytes with the cut undone decode completely: the rule, not the data, removed the tail
    raw_ok = np.concatenate([raw[:int(offs[j + 1])], np.zeros(2, np.uint8), raw[int(offs[j + 1]):]])
    offs_ok = offs.astype(np.int64); offs_ok[j + 1:] += 2
    assert oracle.decode(raw_ok, offs_ok.astype(np.uint32), 1, geom).status == 0

    raw, offs, want2 = malformed.foreign_bank(geom)
    h = oracle.decode(raw, offs, 2, geom)
    assert h.status == oracle.ST_BAD_BANK_SIZE               # in particular no DUPLICATE / foreign words
    e0 = slice(0, int(h.hit_offsets[64])); e1 = slice(int(h.hit_offsets[64]), h.n_hits)
    assert sorted(h.id[e0].astype(np.int64).tolist()) == want2[0]
    assert sorted(h.id[e1].astype(np.int64).tolist()) == want2[1]
    # an event whose end lies in front of its begin loses every bank
    offs_bad = offs.copy(); offs_bad[896] = offs[2 * 896] + 4
    h = oracle.decode(raw, offs_bad, 2, geom)
    assert h.status & oracle.ST_BAD_BANK_SIZE and h.hit_offsets[64] <= len(want2[0])
