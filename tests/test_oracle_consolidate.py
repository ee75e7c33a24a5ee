"""Pins of the track-consolidation oracle against what the definition
fixes: a pure-Python walk, numpy boolean compaction, invariants, and the edge cases."""
import numpy as np

import oracle


def _random_tracks(rng, n_events, mean_tracks, p_keep):
    nt = rng.poisson(mean_tracks, n_events)
    vo = np.concatenate([[0], np.cumsum(nt)]).astype(np.uint32)
    T = int(vo[-1])
    n = np.where(rng.random(T) < p_keep, rng.integers(3, 5, T), 0).astype(np.int32)
    idx = np.where(n[None, :] > 0, rng.integers(0, 10 ** 6, (4, T)), -1).astype(np.int32)
    qop = np.where(n > 0, rng.normal(0, 1e-4, T), 0).astype(np.float32)
    chi2 = np.where(n > 0, rng.random(T) * 20, 0).astype(np.float32)
    return idx, n, qop, chi2, vo


def test_equals_python_walk_and_numpy_mask():
    rng = np.random.default_rng(11)
    idx, n, qop, chi2, vo = _random_tracks(rng, 40, 30.0, 0.6)
    r = oracle.consolidate(idx, n, qop, chi2, vo, 40)
    # (1) pure-Python walk, written independently of the C loop
    keep, offs = [], []
    for e in range(40):
        offs.append(len(keep))
        keep += [t for t in range(int(vo[e]), int(vo[e + 1])) if n[t] > 0]
    offs.append(len(keep))
    assert r.velo_index.tolist() == keep and r.track_offsets.tolist() == offs
    # (2) numpy boolean compaction of every field
    m = n > 0
    assert np.array_equal(r.hit_idx, idx[:, m]) and np.array_equal(r.n_hits, n[m])
    assert np.array_equal(r.qop.view(np.uint32), qop[m].view(np.uint32))
    assert np.array_equal(r.chi2.view(np.uint32), chi2[m].view(np.uint32))
    assert r.status == 0


def test_invariants():
    rng = np.random.default_rng(12)
    idx, n, qop, chi2, vo = _random_tracks(rng, 200, 150.0, 0.8)
    r = oracle.consolidate(idx, n, qop, chi2, vo, 200)
    K = int((n > 0).sum())
    assert r.track_offsets[0] == 0 and r.track_offsets[-1] == K == len(r.velo_index)
    assert np.all(np.diff(r.track_offsets.astype(np.int64)) >= 0)
    assert np.all(np.diff(r.velo_index.astype(np.int64)) > 0)                    # order kept, no duplicates
    ev_of = np.searchsorted(vo, r.velo_index, side="right") - 1                   # event of every kept track
    for e in (0, 17, 199):
        lo, hi = int(r.track_offsets[e]), int(r.track_offsets[e + 1])
        assert np.all(ev_of[lo:hi] == e) and hi - lo == int((n[vo[e]:vo[e + 1]] > 0).sum())
    assert np.all(r.n_hits >= 3)


def test_edge_cases():
    z = lambda dt: np.zeros(0, dt)
    r = oracle.consolidate(np.zeros((4, 0), np.int32), z(np.int32), z(np.float32), z(np.float32),
                           np.zeros(4, np.uint32), 3)                              # events without VELO tracks
    assert r.track_offsets.tolist() == [0, 0, 0, 0] and len(r.velo_index) == 0
    rng = np.random.default_rng(13)
    idx, n, qop, chi2, vo = _random_tracks(rng, 5, 20.0, 1.0)                      # every track kept
    r = oracle.consolidate(idx, n, qop, chi2, vo, 5)
    assert np.array_equal(r.velo_index, np.arange(vo[-1])) and np.array_equal(r.track_offsets, vo)
    n0 = np.zeros_like(n)                                                           # nothing kept
    r = oracle.consolidate(idx, n0, qop, chi2, vo, 5)
    assert len(r.velo_index) == 0 and not r.track_offsets.any()
    r = oracle.consolidate(idx, n, qop, chi2, vo, 5, capacity=7)                    # capacity: offsets stay exact
    assert r.status == 8 and len(r.velo_index) == 7 and np.array_equal(r.track_offsets, vo)
    assert np.array_equal(r.velo_index, np.arange(7))


def test_on_compass_output(wl):
    geom, b, p = wl(2, 20)
    h, t = oracle.run_batch(b, geom, p)
    r = oracle.consolidate(t.hit_idx, t.n_hits, t.qop, t.chi2, b.velo_offsets, b.n_events)
    m = t.n_hits > 0
    assert 0 < m.sum() < m.size
    assert np.array_equal(r.velo_index, np.nonzero(m)[0]) and np.array_equal(r.hit_idx, t.hit_idx[:, m])
