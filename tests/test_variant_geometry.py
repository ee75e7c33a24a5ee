"""The oracle on the second, non-uniform geometry (synth/variant.py: finer inner columns and rows, rows that
overlap in y, per-sector z, a 4096-entry raw-id table, optionally shuffled rows): the same pins that do not
depend on the regular layout, so that the GPU parity tests on this geometry compare against a checked oracle."""
import numpy as np
import pytest

import oracle
import synth
from synth import variant as V
from synth.events import EventModel

MODEL = EventModel(mean_tracks=60.0, efficiency=0.97, noise_mean=700.0)


@pytest.fixture(scope="module", params=[False, True], ids=["rows_sorted", "rows_shuffled"])
def vwl(request):
    geom = V.make_staggered_geometry(shuffle_rows=request.param)
    return geom, V.generate_batch_tables(geom, MODEL, seed=21, n_events=12)


def test_geometry_contract(vwl):
    geom, _ = vwl
    assert geom.n_sectors == 896 and geom.n_groups == 56 and geom.id_table_size == 4096
    assert np.all(np.diff(geom.sector_group.astype(np.int64)) >= 0)
    assert len(np.unique(geom.pitch)) == 2 and len(np.unique(geom.z)) == 8          # two pitches, staggered z
    for g in range(geom.n_groups):
        s = slice(int(geom.group_first_sector[g]), int(geom.group_first_sector[g + 1]))
        assert len(np.unique(geom.dxdy[s])) == 1 and s.stop - s.start == 16


def test_decode_invariants_and_round_trip(vwl):
    geom, b = vwl
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    assert h.status == 0 and h.n_hits == b.total_hits
    ng = geom.n_groups
    for e in range(b.n_events):
        for g in range(ng):
            lo, hi = int(h.hit_offsets[e * ng + g]), int(h.hit_offsets[e * ng + g + 1])
            x = h.x_at_y0[lo:hi]
            assert np.all(np.diff(x) >= 0)
            assert np.all(x >= geom.group_xmin[g]) and np.all(x <= geom.group_xmax[g])
            sec = geom.id_to_sector[h.id[lo:hi] >> 9]
            assert np.all(geom.sector_group[sec] == g)
            assert np.array_equal(h.z_at_y0[lo:hi], geom.z[sec]) and np.array_equal(h.y_end[lo:hi], geom.y_end[sec])
    # closed form of x in float64 (within 1 ulp of fp32), strip recovered from the id
    sec = geom.id_to_sector[h.id[:h.n_hits] >> 9]
    strip = (h.id[:h.n_hits] & 0x1FF).astype(np.float64)
    x64 = geom.x0[sec].astype(np.float64) + (strip + 0.25) * geom.pitch[sec].astype(np.float64)
    dx = h.x_at_y0[:h.n_hits].astype(np.float64) - x64
    half = 0.5 * geom.pitch[sec].astype(np.float64)
    assert np.all((np.abs(dx) < 1e-3) | (np.abs(dx - half) < 1e-3))                   # frac = 0 or 1


def test_window_search_equals_linear_scan_and_finds_tracks(vwl):
    geom, b = vwl
    p = synth.make_compass_params()
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    args = (h, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, geom, p)
    t0, t1 = oracle.compass(*args, mode=0), oracle.compass(*args, mode=1)
    assert np.array_equal(t0.cand_n, t1.cand_n) and np.array_equal(t0.cand_list, t1.cand_list)     # BF-1
    assert np.array_equal(t0.hit_idx, t1.hit_idx) and np.array_equal(t0.chi2.view(np.uint32), t1.chi2.view(np.uint32))
    assert (t0.n_hits == 4).sum() > 50 and (t0.n_hits == 3).sum() > 5
    # the row overlap is exercised: some track has two candidates with identical x in one layer group
    assert (t0.cand_n.max(axis=1) >= 2).any()
