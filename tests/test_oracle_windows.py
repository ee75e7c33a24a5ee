"""Pins of the paper-literal window ranges (Fig. 7) and of the tracklet
search that starts from them.  None re-calls the oracle's own search: the ranges are checked against a numpy
linear scan, against the BF-1 candidate lists of the fused definition, and by their own invariants."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth


def _resid32(h, idx, x_e, y_e):
    """d of DESIGN.md section 3 in float32, vectorised over hits (numpy float32 ops round like the oracle's)."""
    F = np.float32
    return (h.x_at_y0[idx] + h.dxdy[idx] * F(y_e)).astype(np.float32) - F(x_e)


def _extrap(b, geom, t, l):
    F = np.float32
    dzv = F(geom.layer_z[l]) - F(b.velo_z)
    return F(b.velo_x[t] + F(b.velo_tx[t] * dzv)), F(b.velo_y[t] + F(b.velo_ty[t] * dzv))


@pytest.mark.parametrize("config,n", [(2, 12), (4, 3)])
def test_ranges_are_the_windows_of_a_linear_scan(wl, config, n):
    """Every stored range is exactly the set of hits of ITS group with |d| <= win_half (numpy scan of the group),
    (-1, -1) where that set is empty; layout = W begins then W sizes per panel; W = 1, 3, 5 are nested."""
    geom, b, p = wl(config, n)
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    wins = {W: oracle.search_windows(h, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events,
                                     geom, p, W)[0] for W in (1, 3, 5)}
    ev = np.repeat(np.arange(b.n_events), np.diff(b.velo_offsets.astype(np.int64)))
    gpl = geom.n_groups // 4
    n_ranges = 0
    for t in range(0, b.n_velo_total, 7):
        goff = h.hit_offsets[ev[t] * geom.n_groups:(ev[t] + 1) * geom.n_groups + 1].astype(np.int64)
        for l in range(4):
            x_e, y_e = _extrap(b, geom, t, l)
            c = np.float32(x_e - np.float32(geom.layer_dxdy[l] * y_e))
            ge = np.nonzero(geom.group_xmax[l * gpl:(l + 1) * gpl] >= c)[0]
            central = l * gpl + (int(ge[0]) if ge.size else gpl - 1)
            for W in (1, 3, 5):
                w = wins[W][t, l]
                groups = [central + o for o in (0, -1, 1, -2, 2)[:W]]
                for k, g in enumerate(groups):
                    if g < l * gpl or g >= (l + 1) * gpl:
                        assert (w[k], w[W + k]) == (-1, -1)
                        continue
                    idx = np.arange(goff[g], goff[g + 1])
                    inside = idx[np.abs(_resid32(h, idx, x_e, y_e)) <= np.float32(p.win_half[l])]
                    if inside.size == 0:
                        assert (w[k], w[W + k]) == (-1, -1)
                    else:
                        assert np.array_equal(inside, np.arange(inside[0], inside[-1] + 1))      # one contiguous run
                        assert (w[k], w[W + k]) == (inside[0] - goff[0], inside.size)
                        n_ranges += 1
            assert np.array_equal(wins[3][t, l][[0, 3]], wins[1][t, l])                      # nested, same central slot
            assert np.array_equal(wins[5][t, l][[0, 1, 2, 5, 6, 7]], wins[3][t, l])
    assert n_ranges > 500


@pytest.mark.parametrize("config,n", [(1, None), (2, 25), (4, 4)])
def test_five_sectors_equal_the_exact_window(wl, config, n):
    """With 5 sector groups every group a window of these configs can touch is searched: the hits of the ranges that
    pass the y test are the linear-scan candidate lists (BF-1), and the tracklets are those of the fused definition
    bit for bit.  1 and 3 sectors give subsets."""
    geom, b, p = wl(config, n)
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    big = dataclasses.replace(p, max_candidates_per_layer=4096)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, geom)
    bf1 = oracle.compass(h, *args, big, mode=1)
    ref = oracle.compass(h, *args, p, mode=0)
    counts = {}
    for W in (1, 3, 5):
        win, st = oracle.search_windows(h, *args, p, W)
        assert st == 0
        t = oracle.compass_from_windows(h, win, *args, p, W)
        counts[W] = t.cand_n
        if W == 5:
            assert np.array_equal(t.cand_n, bf1.cand_n)
            assert np.array_equal(t.hit_idx, ref.hit_idx) and np.array_equal(t.n_hits, ref.n_hits)
            assert np.array_equal(t.chi2.view(np.uint32), ref.chi2.view(np.uint32))
            assert np.array_equal(t.qop.view(np.uint32), ref.qop.view(np.uint32))
    assert np.all(counts[1] <= counts[3]) and np.all(counts[3] <= counts[5])
    if config != 1:
        assert (counts[1] < counts[5]).any()                    # one sector really misses hits


def test_windows_edge_cases(geom):
    from synth.events import EventModel, generate_batch, generate_event, assemble_batch
    p = synth.make_compass_params()
    b = generate_batch(geom, EventModel(fixed_tracks=6, noise_mean=0.0, efficiency=0.0), seed=3, n_events=2)   # no hits
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    win, st = oracle.search_windows(h, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, 2, geom, p, 3)
    assert st == 0 and win.shape == (12, 4, 6) and np.all(win == -1)
    # an event of more than 32767 hits cannot be indexed by shorts: flagged, every range empty
    big = assemble_batch(geom, [generate_event(geom, EventModel(fixed_tracks=5, noise_mean=40000.0), 4, 0)])
    h = oracle.decode(big.raw, big.bank_offsets, 1, geom, big.hit_capacity)
    assert h.n_hits > 32767
    win, st = oracle.search_windows(h, big.velo_x, big.velo_y, big.velo_tx, big.velo_ty, big.velo_z, big.velo_offsets, 1,
                                    geom, p, 5)
    assert st == 32 and np.all(win == -1)
