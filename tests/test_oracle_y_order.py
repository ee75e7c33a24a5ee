"""Pins of the paper's literal Y order inside a sector group (
DESIGN.md A25): decode with order "y" and the window search by binary searches over Y."""
import numpy as np
import pytest

import oracle
import synth
from synth import geometry as G
from synth import variant as V
from synth.events import EventModel, encode_event


def _geoms():
    return {"regular": synth.make_geometry(), "staggered": V.make_staggered_geometry(),
            "staggered_shuffled_rows": V.make_staggered_geometry(shuffle_rows=True)}


def _batch(name, geom, n=12):
    if name == "regular":
        return synth.events.generate_batch(geom, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), 17, n)
    return V.generate_batch_tables(geom, EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0), seed=17, n_events=n)


@pytest.mark.parametrize("name", ["regular", "staggered", "staggered_shuffled_rows"])
def test_y_order_is_a_stable_resort_of_the_x_order(name):
    """Same hits, same offsets; inside every group the Y order equals numpy's stable lexsort of the x-ordered
    container by (y_begin, x) (an independent sort routine applied to the pinned x order)."""
    geom = _geoms()[name]
    b = _batch(name, geom)
    hx = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity, order="x")
    hy = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity, order="y")
    assert hy.status == hx.status == 0 and np.array_equal(hx.hit_offsets, hy.hit_offsets)
    n = hx.n_hits
    grp = np.repeat(np.arange(hx.hit_offsets.size - 1), np.diff(hx.hit_offsets.astype(np.int64)))
    perm = np.lexsort((hx.x_at_y0[:n], hx.y_begin[:n], grp))            # stable; last key is the primary one
    for f in oracle.Hits.FIELDS:
        assert np.array_equal(getattr(hy, f)[:n], getattr(hx, f)[:n][perm]), f
    # the sort key really is non-decreasing, and x inside a row
    same = grp[1:] == grp[:-1]
    yb, x = hy.y_begin[:n], hy.x_at_y0[:n]
    assert np.all(yb[1:][same] >= yb[:-1][same])
    row = same & (yb[1:] == yb[:-1])
    assert np.all(x[1:][row] >= x[:-1][row])
    assert (perm != np.arange(n)).sum() > n // 2                        # it is a different order


def test_y_order_ties_keep_the_fill_order(geom):
    """Hand-built: two rows of one X-layer column with identical strips, words given out of order.  Y order = row by
    row; inside a row ascending strip; the x order interleaves the rows instead."""
    s_lo, s_hi = G.dense_sector(0, 4, 3), G.dense_sector(0, 4, 9)
    sector = [s_hi, s_lo, s_hi, s_lo, s_lo, s_hi]
    strip = [300, 300, 20, 20, 400, 400]
    raw, offs = encode_event(geom, np.asarray(sector), np.asarray(strip), np.zeros(6, int), np.zeros(6, int), None)
    hy = oracle.decode(raw, offs.astype(np.uint32), 1, geom, order="y")
    hx = oracle.decode(raw, offs.astype(np.uint32), 1, geom, order="x")
    rid = lambda s: int(geom.sector_raw_id[s]) << 9
    assert hy.id[:6].tolist() == [rid(s_lo) | 20, rid(s_lo) | 300, rid(s_lo) | 400, rid(s_hi) | 20, rid(s_hi) | 300, rid(s_hi) | 400]
    assert hx.id[:6].tolist() == [rid(s_lo) | 20, rid(s_hi) | 20, rid(s_lo) | 300, rid(s_hi) | 300, rid(s_lo) | 400, rid(s_hi) | 400]


@pytest.mark.parametrize("name", ["regular", "staggered", "staggered_shuffled_rows"])
def test_y_window_search_equals_linear_scan(name):
    """BF-1 for the Y order: candidates found through the two binary searches over Y equal the linear scan of the
    layer, and the tracklets carry the same hits (by id) as on the x-ordered container wherever no exact tie decides."""
    geom = _geoms()[name]
    b = _batch(name, geom, 10)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, geom)
    hy = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity, order="y")
    for p in (synth.make_compass_params(), synth.make_compass_params(window_scale=2.0, max_candidates_per_layer=4)):
        t3 = oracle.compass(hy, *args, p, mode=3)
        t1 = oracle.compass(hy, *args, p, mode=1)
        assert np.array_equal(t3.cand_n, t1.cand_n) and np.array_equal(t3.cand_list, t1.cand_list)
        assert np.array_equal(t3.hit_idx, t1.hit_idx) and np.array_equal(t3.chi2.view(np.uint32), t1.chi2.view(np.uint32))
        assert (t3.n_hits > 0).sum() > 500
    # against the x-ordered container: same physics
    hx = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity, order="x")
    p = synth.make_compass_params(max_candidates_per_layer=32)
    tx, ty = oracle.compass(hx, *args, p, mode=0), oracle.compass(hy, *args, p, mode=3)
    idx, idy = np.where(tx.hit_idx >= 0, hx.id[np.maximum(tx.hit_idx, 0)], -1), np.where(ty.hit_idx >= 0, hy.id[np.maximum(ty.hit_idx, 0)], -1)
    same = np.all(idx == idy, axis=0)
    assert same.mean() > 0.999 and np.array_equal(tx.n_hits, ty.n_hits)
    assert np.array_equal(tx.chi2.view(np.uint32), ty.chi2.view(np.uint32))
