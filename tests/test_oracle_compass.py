"""Pins of the Compass oracle.  The oracle is compared with things other
than itself: a float64 lstsq-based brute force, closed forms, hand-built predicates, generator truth."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth
from synth import geometry as G
from synth.events import EventModel, generate_batch, KAPPA, Z_MAG, Z_VELO
from helpers import make_hits, run_one, brute_force64

W = 12.0 / G.PITCH ** 2


def run(b, geom, p, mode=0, hits=None):
    h = hits or oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    return h, oracle.compass(h, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events,
                             geom, p, mode)


def same_tracks(a, b):
    assert np.array_equal(a.hit_idx, b.hit_idx)
    assert np.array_equal(a.n_hits, b.n_hits)
    assert np.array_equal(a.qop.view(np.uint32), b.qop.view(np.uint32))
    assert np.array_equal(a.chi2.view(np.uint32), b.chi2.view(np.uint32))


# ---- BF-1: binary-search windows == linear scan of the layer, exactly --------------------------------
@pytest.mark.parametrize("cfg,n,over", [(1, None, {}), (2, None, {}), (2, 30, dict(max_candidates_per_layer=4)),
                                        (2, 30, dict(window_scale=2.0, max_candidates_per_layer=8)),
                                        (4, 4, {})])
def test_bf1_window_equals_linear_scan(wl, cfg, n, over):
    geom, b, p = wl(cfg, n)
    if over:
        p = synth.CONFIGS[cfg].compass_params(**over)
    h, t0 = run(b, geom, p, 0)
    _, t1 = run(b, geom, p, 1, hits=h)
    assert np.array_equal(t0.cand_n, t1.cand_n)
    assert np.array_equal(t0.cand_list, t1.cand_list)
    same_tracks(t0, t1)
    if over.get("max_candidates_per_layer", 99) <= 8:
        assert (t0.cand_n > p.max_candidates_per_layer).any()        # the cap is exercised
        full = (t0.cand_list >= 0).sum(axis=2)
        assert np.array_equal(full, np.minimum(t0.cand_n, p.max_candidates_per_layer))
        cl = t0.cand_list.astype(np.int64)
        both = (cl[:, :, 1:] >= 0) & (cl[:, :, :-1] >= 0)
        assert np.all(np.diff(cl, axis=2)[both] > 0)                     # list stays in ascending h


# ---- BF-2: seeded search == exhaustive enumeration ---------------------------------------------------
def test_bf2_seeded_equals_exhaustive_config1(wl):
    geom, b, p = wl(1)
    h, t0 = run(b, geom, p, 0)
    _, t2 = run(b, geom, p, 2, hits=h)
    same_tracks(t0, t2)
    assert (t0.n_hits > 0).sum() >= 10


def test_bf2_seeded_equals_exhaustive_small_noisy(geom):
    m = EventModel(fixed_tracks=8, efficiency=0.9, noise_mean=60.0)
    b = generate_batch(geom, m, seed=21, n_events=25)
    p = synth.make_compass_params(max_candidates_per_layer=64, window_scale=2.0)
    h, t0 = run(b, geom, p, 0)
    _, t2 = run(b, geom, p, 2, hits=h)
    same_tracks(t0, t2)
    assert (t0.n_hits == 3).any() and (t0.n_hits == 4).any()


def test_float64_lstsq_brute_force(geom):
    """Independent float64 implementation (np.linalg.lstsq fit, plain loops) on tiny events."""
    m = EventModel(fixed_tracks=6, efficiency=0.9, noise_mean=40.0)
    b = generate_batch(geom, m, seed=33, n_events=12)
    p = synth.make_compass_params(max_candidates_per_layer=64)
    h, t = run(b, geom, p, 0)
    n_cmp = 0
    for e in range(b.n_events):
        lo, hi = int(h.hit_offsets[e * 64]), int(h.hit_offsets[(e + 1) * 64])
        for k in range(int(b.velo_offsets[e]), int(b.velo_offsets[e + 1])):
            ref = brute_force64(h, lo, hi, geom, p, float(b.velo_x[k]), float(b.velo_y[k]), float(b.velo_tx[k]),
                                float(b.velo_ty[k]))
            if ref is None:
                assert t.n_hits[k] == 0 and np.all(t.hit_idx[:, k] == -1) and t.qop[k] == 0 and t.chi2[k] == 0
                continue
            # skip results decided by a float64-vs-float32 hair (none expected, but be explicit)
            if np.isfinite(t.runner_chi2[k]) and abs(t.runner_chi2[k] - t.chi2[k]) <= 1e-4 * t.chi2[k]:
                continue
            assert tuple(t.hit_idx[:, k]) == ref[0] and t.n_hits[k] == ref[1]
            assert t.chi2[k] == pytest.approx(ref[2], rel=2e-3, abs=1e-4)
            assert t.qop[k] == pytest.approx(ref[3], rel=1e-4, abs=1e-9)
            n_cmp += 1
    assert n_cmp >= 40


# ---- fit ---------------------------------------------------------------------------------------------
def test_fit_equals_weighted_lstsq(geom):
    p = synth.make_compass_params()
    rng = np.random.default_rng(0)
    for trial in range(200):
        n = int(rng.integers(3, 5))
        layers = np.sort(rng.choice(4, n, replace=False))
        z = np.asarray(G.LAYER_Z)[layers]
        b_true = rng.uniform(-0.03, 0.03)
        d = b_true * (z - Z_MAG) + rng.normal(0, 0.06, n)
        w = np.full(n, W)
        a, b, chi2, qop = oracle.fit(d, z, w, p)
        dz = np.concatenate([[0.0], np.float32(z).astype(np.float64) - Z_MAG])
        dd = np.concatenate([[0.0], np.float32(d).astype(np.float64)])
        ww = np.concatenate([[p.w_velo], w])
        A = np.stack([np.ones(n + 1), dz], 1) * np.sqrt(ww)[:, None]
        sol, *_ = np.linalg.lstsq(A, dd * np.sqrt(ww), rcond=None)
        chi64 = float((ww * (dd - sol[0] - sol[1] * dz) ** 2).sum())
        assert a == pytest.approx(sol[0], abs=2e-4)
        assert b == pytest.approx(sol[1], rel=1e-4, abs=1e-7)
        assert chi2 == pytest.approx(chi64, rel=1e-2, abs=2e-4)
        assert qop == pytest.approx(sol[1] / KAPPA, rel=1e-4, abs=1e-9)


def test_fit_collinear_exact(geom):
    p = synth.make_compass_params()
    z = np.asarray(G.LAYER_Z)
    b_true = 2.0 ** -6                                   # exactly representable slope, dz are multiples of 0.5
    d = b_true * (z - Z_MAG)
    a, b, chi2, qop = oracle.fit(d, z, np.full(4, W), p)
    assert abs(a) < 1e-4 and b == pytest.approx(b_true, rel=1e-6) and chi2 < 1e-4
    assert qop == pytest.approx(b_true / 60.0, rel=1e-6)
    # sign convention: positive slope in d  <=>  positive q/p
    a, b, chi2, qop = oracle.fit(-d[:3], z[:3], np.full(3, W), p)
    assert qop < 0 and chi2 < 1e-4
    # an offset common to all hits is NOT absorbed: the VELO pseudo-point pins the line at z_mag
    a, b, chi2, qop = oracle.fit(d + 1.0, z, np.full(4, W), p)
    assert chi2 > 20.0


# ---- hand-built predicates ---------------------------------------------------------------------------
def straight_track_hits(b_slope, x_off=(0, 0, 0, 0), y=100.0, x_v=200.0, present=(1, 1, 1, 1)):
    """Hits for a VELO track x = x_v (tx = ty = 0), y = y: residual d_l = b*(z_l - z_mag) + x_off[l]."""
    per = [[], [], [], []]
    for l in range(4):
        if present[l]:
            d = b_slope * (G.LAYER_Z[l] - Z_MAG) + x_off[l]
            x_at_y = x_v + d                               # hit x at the track's y
            per[l].append((x_at_y - G.LAYER_DXDY[l] * y, 96.0, 192.0))
    return per


VELO = [(200.0, 100.0, 0.0, 0.0)]


def test_recovers_a_kicked_track(geom):
    p = synth.make_compass_params()
    hits = make_hits(geom, straight_track_hits(0.01))
    t = run_one(hits, geom, p, VELO)
    assert t.n_hits[0] == 4 and sorted(t.hit_idx[:, 0]) == [0, 1, 2, 3]
    assert t.qop[0] == pytest.approx(0.01 / 60.0, rel=1e-3) and t.chi2[0] < 0.1
    # layer l's index lands in row l
    z_of = hits.z_at_y0[t.hit_idx[:, 0]]
    assert np.array_equal(z_of, np.float32(G.LAYER_Z))


@pytest.mark.parametrize("present,expect_n", [((1, 1, 1, 1), 4), ((1, 0, 1, 1), 3), ((1, 1, 1, 0), 3),
                                              ((0, 1, 1, 1), 3), ((1, 1, 0, 1), 3),     # backward seeds (L3, L1)
                                              ((1, 0, 1, 0), 0), ((0, 1, 0, 1), 0), ((1, 1, 0, 0), 0)])
def test_directions_and_min_hits(geom, present, expect_n):
    hits = make_hits(geom, straight_track_hits(-0.008, present=present))
    for mh in (3, 4):
        p = synth.make_compass_params(min_hits=mh)
        t = run_one(hits, geom, p, VELO)
        want = expect_n if expect_n >= mh else 0
        assert t.n_hits[0] == want
        assert (t.hit_idx[:, 0] >= 0).sum() == want
        if want:
            assert t.qop[0] == pytest.approx(-0.008 / 60.0, rel=2e-3)
            assert np.array_equal(t.hit_idx[:, 0] >= 0, np.asarray(present, bool))
        else:
            assert t.qop[0] == 0 and t.chi2[0] == 0


def test_window_and_y_edges(geom):
    p = synth.make_compass_params()
    D0 = p.win_half[0]
    for off, inside in ((D0 - 0.01, True), (D0 + 0.01, False), (-D0 + 0.01, True), (-D0 - 0.01, False)):
        hits = make_hits(geom, [[(200.0 + off, 96.0, 192.0)], [], [], []])
        t = run_one(hits, geom, p, VELO)
        assert t.cand_n[0, 0] == (1 if inside else 0)
    for yb, ye, inside in ((100.4, 192.0, True), (100.6, 192.0, False), (0.0, 99.6, True), (0.0, 99.4, False)):
        hits = make_hits(geom, [[(200.0, yb, ye)], [], [], []])
        t = run_one(hits, geom, p, VELO)
        assert t.cand_n[0, 0] == (1 if inside else 0)
    # stereo layer: d uses x_at_y0 + dxdy * y_e
    hits = make_hits(geom, [[], [(200.0 - G.TAN5 * 100.0 + 3.0, 96.0, 192.0)], [], []])
    t = run_one(hits, geom, p, VELO)
    assert t.cand_n[0, 1] == 1
    hits = make_hits(geom, [[], [(200.0 + G.TAN5 * 100.0 + 3.0, 96.0, 192.0)], [], []])   # wrong sign of the stereo term
    t = run_one(hits, geom, p, VELO)
    assert t.cand_n[0, 1] == 0
    # extrapolation: x_e = x_v + tx * (z_l - 770)
    hits = make_hits(geom, [[(200.0 + 0.1 * (2327.5 - 770.0), 96.0, 400.0)], [], [], []])
    t = run_one(hits, geom, p, [(200.0, 100.0, 0.1, 0.05)])
    assert t.cand_n[0, 0] == 1 and t.cand_list[0, 0, 0] == 0


def test_seed_cuts(geom):
    p = synth.make_compass_params()
    # kink cut: all hits shifted by a common 3 mm offset -> slope fine, intercept at z_mag = 3 > 1.5
    hits = make_hits(geom, straight_track_hits(0.005, x_off=(3, 3, 3, 3)))
    assert run_one(hits, geom, p, VELO).n_hits[0] == 0
    hits = make_hits(geom, straight_track_hits(0.005, x_off=(1, 1, 1, 1)))
    t = run_one(hits, geom, p, VELO)
    assert t.n_hits[0] == 0 or t.chi2[0] > 20          # passes the kink cut, killed by chi2 (w_velo * 1^2 = 100)
    # slope cut: hits inside the windows but on a line steeper than max_slope through a far intercept
    p2 = dataclasses.replace(p, kink_tol=1e9, max_chi2_ndf=1e9)
    steep = [(-15.0 if l < 2 else 15.0) for l in range(4)]      # slope ~ 30/270 = 0.11 >> 0.0315
    hits = make_hits(geom, straight_track_hits(0.0, x_off=steep))
    assert run_one(hits, geom, p2, VELO).n_hits[0] == 0
    # seed tolerance: L1 hit 0.6 mm off the seed line is not compatible, 0.4 mm is
    for off, n in ((0.6, 3), (0.4, 4)):
        hits = make_hits(geom, straight_track_hits(0.01, x_off=(0, off, 0, 0)))
        p3 = dataclasses.replace(p, max_chi2_ndf=1e9)
        t = run_one(hits, geom, p3, VELO)
        assert t.n_hits[0] == n
        if n == 3:
            assert t.hit_idx[1, 0] == -1


def test_prefers_four_hits_then_lowest_chi2(geom):
    p = synth.make_compass_params()
    per = straight_track_hits(0.01)
    # a second, worse L1 hit (0.3 mm off) and a second, worse L3 hit
    d1 = 0.01 * (G.LAYER_Z[1] - Z_MAG) + 0.3
    per[1].append((200.0 + d1 - G.LAYER_DXDY[1] * 100.0, 96.0, 192.0))
    d3 = 0.01 * (G.LAYER_Z[3] - Z_MAG) - 0.25
    per[3].append((200.0 + d3, 96.0, 192.0))
    hits = make_hits(geom, per)
    t = run_one(hits, geom, p, VELO)
    assert t.n_hits[0] == 4 and t.n_fits[0] == 8          # (2+1)*(2+1) - 1 combos with >= 3 hits
    sel = t.hit_idx[:, 0]
    d_sel = hits.x_at_y0[sel] + hits.dxdy[sel] * np.float32(100.0) - np.float32(200.0)
    assert np.allclose(d_sel, 0.01 * (np.asarray(G.LAYER_Z) - Z_MAG), atol=1e-3)     # the on-line hits win
    assert np.isfinite(t.runner_chi2[0]) and t.runner_chi2[0] > t.chi2[0]
    # exact tie: duplicate of the L1 hit -> lower hit index wins, runner-up chi2 equals chi2
    per = straight_track_hits(0.01)
    per[1].append(per[1][0])
    hits = make_hits(geom, per)
    t = run_one(hits, geom, p, VELO)
    assert t.runner_chi2[0] == t.chi2[0]
    l1 = [h for h in range(hits.n_hits) if hits.z_at_y0[h] == np.float32(G.LAYER_Z[1])]
    assert t.hit_idx[1, 0] == min(l1)


def test_candidate_cap_keeps_closest(geom):
    p = synth.make_compass_params(max_candidates_per_layer=3)
    offs = [-6.0, -2.0, -0.5, 0.2, 2.0, 5.0, 7.0]
    hits = make_hits(geom, [[(200.0 + o, 96.0, 192.0) for o in offs], [], [], []])
    t = run_one(hits, geom, p, VELO)
    assert t.cand_n[0, 0] == 7
    kept = t.cand_list[0, 0]
    assert np.allclose(np.sort(hits.x_at_y0[kept] - 200.0), [-2.0, -0.5, 0.2], atol=1e-4)
    assert np.all(np.diff(kept) > 0)
    # tie in |d|: lower hit index wins
    hits = make_hits(geom, [[(198.0, 96.0, 192.0), (202.0, 96.0, 192.0), (200.5, 96.0, 192.0)], [], [], []])
    p1 = synth.make_compass_params(max_candidates_per_layer=2)
    t = run_one(hits, geom, p1, VELO)
    assert sorted(t.cand_list[0, 0].tolist()) == [0, 1]        # x-sorted: 198 -> 0, 200.5 -> 1, 202 -> 2


# ---- truth, charge, monotonicity ------------------------------------------------------------------------
def test_charge_sign_and_momentum(wl):
    geom, b, p = wl(2)
    h, t = run(b, geom, p)
    idx = t.hit_idx.T
    ids = np.where(idx >= 0, h.id[np.clip(idx, 0, None)].astype(np.int64), -2)
    all_true = (t.n_hits >= 3) & np.all((ids == b.truth_hit_id) | (idx < 0), axis=1)
    assert all_true.sum() > 8000
    r = t.qop[all_true].astype(np.float64) * b.truth_p[all_true] * b.truth_q[all_true]
    assert np.all(r > 0)                                              # sign = generated charge, always
    lowp = b.truth_p[all_true] < 3000
    assert np.sqrt(((r[lowp] - 1) ** 2).mean()) < 0.01                # ~0.35 % at 2-3 GeV
    assert abs(np.median(r) - 1) < 0.01
    m = synth.physics_metrics(b.truth_hit_id, b.truth_q, h.id, t.hit_idx, t.n_hits, t.qop)
    assert m["efficiency"] > 0.97 and m["ghost_rate"] < 0.08 and m["charge_ok"] == 1.0


def test_truth_recovery_noise_free_isolated(geom):
    m = EventModel(fixed_tracks=20, efficiency=1.0, noise_mean=0.0)
    b = generate_batch(geom, m, seed=1, n_events=60)
    p = synth.make_compass_params()
    h, t = run(b, geom, p)
    idx = t.hit_idx.T
    ids = np.where(idx >= 0, h.id[np.clip(idx, 0, None)].astype(np.int64), -1)
    n_true = (b.truth_hit_id >= 0).sum(axis=1)
    # isolated = no foreign hit among the track's candidates: candidates per layer == own hit present
    isolated = np.all(t.cand_n == (b.truth_hit_id >= 0), axis=1)
    sel = isolated & (n_true >= 3)
    assert sel.sum() > 500
    assert np.array_equal(ids[sel], b.truth_hit_id[sel])             # exactly its true hits
    assert np.array_equal(t.n_hits[sel], n_true[sel])
    # tracks with < 3 true hits and nothing foreign: no tracklet
    none = isolated & (n_true < 3)
    assert none.sum() > 50 and np.all(t.n_hits[none] == 0)
    # the non-isolated remainder is reported, not asserted
    rest = ~isolated & (n_true >= 3)
    assert (ids[rest] == b.truth_hit_id[rest]).all(axis=1).mean() > 0.7


def test_monotonic_in_candidates_and_min_hits(wl):
    geom, b, _ = wl(2, 40)
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    prev = None
    for C in (1, 2, 4, 8, 16, 32):
        p = synth.make_compass_params(max_candidates_per_layer=C)
        _, t = run(b, geom, p, hits=h)
        if prev is not None:
            # raising C never worsens (n, -chi2): candidate sets are nested (A7)
            worse = (t.n_hits < prev.n_hits) | ((t.n_hits == prev.n_hits) & (t.n_hits > 0) & (t.chi2 > prev.chi2))
            # forward-first rule (A11) can swap a backward result for a forward one: only then may chi2 rise
            fwd_new = (t.hit_idx[0] >= 0) & (t.hit_idx[2] >= 0)
            fwd_old = (prev.hit_idx[0] >= 0) & (prev.hit_idx[2] >= 0)
            assert not (worse & ~(fwd_new & ~fwd_old)).any()
        prev = t
    p3 = synth.make_compass_params(min_hits=3)
    p4 = synth.make_compass_params(min_hits=4)
    _, t3 = run(b, geom, p3, hits=h)
    _, t4 = run(b, geom, p4, hits=h)
    four = t3.n_hits == 4
    assert four.sum() > 1000
    assert np.array_equal(t3.hit_idx[:, four], t4.hit_idx[:, four])
    assert np.array_equal(t3.chi2[four], t4.chi2[four])
    assert np.all((t4.n_hits == 4) | (t4.n_hits == 0))


def test_velo_permutation_equivariance(wl):
    geom, b, p = wl(2, 10)
    h, t = run(b, geom, p)
    rng = np.random.default_rng(9)
    perm = np.concatenate([rng.permutation(np.arange(b.velo_offsets[e], b.velo_offsets[e + 1]))
                           for e in range(b.n_events)]).astype(np.int64)
    t2 = oracle.compass(h, b.velo_x[perm], b.velo_y[perm], b.velo_tx[perm], b.velo_ty[perm], b.velo_z,
                        b.velo_offsets, b.n_events, geom, p)
    assert np.array_equal(t2.hit_idx, t.hit_idx[:, perm])
    assert np.array_equal(t2.chi2, t.chi2[perm]) and np.array_equal(t2.qop, t.qop[perm])


def test_event_chunks_equal_whole(wl):
    geom, b, p = wl(2, 20)
    h, t = run(b, geom, p)
    T = b.n_velo_total
    out = oracle.Tracks(np.full((4, T), -1, np.int32), np.zeros(T, np.int32), np.zeros(T, np.float32),
                        np.zeros(T, np.float32), np.full(T, np.inf, np.float32), np.zeros((T, 4), np.int32),
                        np.full((T, 4, p.max_candidates_per_layer), -1, np.int32), np.zeros(T, np.int32))
    for lo, n in ((0, 7), (7, 8), (15, 5)):
        oracle.compass_into(out, h, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets,
                            b.n_events, geom, p, 0, first_event=lo, n_sub=n)
    same_tracks(out, t)


def test_no_tracks_and_empty_events(geom):
    m = EventModel(fixed_tracks=0, noise_mean=50.0)
    b = generate_batch(geom, m, seed=2, n_events=3)
    p = synth.make_compass_params()
    h, t = run(b, geom, p)
    assert t.n_hits.shape == (0,) and t.hit_idx.shape == (4, 0)
    m = EventModel(fixed_tracks=5, noise_mean=0.0, efficiency=0.0)
    b = generate_batch(geom, m, seed=2, n_events=2)
    h, t = run(b, geom, p)
    assert h.n_hits == 0 and np.all(t.n_hits == 0) and np.all(t.hit_idx == -1)


def test_golden_config1(wl):
    """Regression fixture written by tests/golden/make_golden.py (oracle only; see its docstring)."""
    import os
    geom, b, p = wl(1)
    h, t = oracle.run_batch(b, geom, p)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_oracle.txt")
    nH = nT = 0
    for line in open(path):
        f = line.split()
        if f[0] == "H":
            k = int(f[1]); nH += 1
            assert int(h.id[k]) == int(f[2]) and int(h.x_at_y0[k:k + 1].view(np.uint32)[0]) == int(f[3], 16)
        elif f[0] == "T":
            k = int(f[1]); nT += 1
            assert int(t.n_hits[k]) == int(f[2]) and [int(v) for v in t.hit_idx[:, k]] == [int(v) for v in f[3:7]]
            assert int(t.qop[k:k + 1].view(np.uint32)[0]) == int(f[7], 16)
            assert int(t.chi2[k:k + 1].view(np.uint32)[0]) == int(f[8], 16)
    assert nH == h.n_hits and nT == 20


# ---- best of both seed directions ------------------------------------------------
def test_both_directions_mode(geom):
    """both_directions = 1: (a) equals the float64 brute force taking the better of the two directions,
    (b) is never worse than the A11 result in (n, chi2), identical wherever forward alone decided and backward
    has nothing better, (c) seeded search == exhaustive search (BF-2) in this mode too."""
    import dataclasses
    m = EventModel(fixed_tracks=8, efficiency=0.85, noise_mean=60.0)
    b = generate_batch(geom, m, seed=41, n_events=15)
    p0 = synth.make_compass_params(max_candidates_per_layer=64)
    p1 = dataclasses.replace(p0, both_directions=1)
    h, t0 = run(b, geom, p0, 0)
    _, t1 = run(b, geom, p1, 0)
    _, t1x = run(b, geom, p1, 2)
    assert np.array_equal(t1.hit_idx, t1x.hit_idx) and np.array_equal(t1.chi2.view(np.uint32), t1x.chi2.view(np.uint32))
    assert np.array_equal(t0.n_hits > 0, t1.n_hits > 0)
    assert np.all(t1.n_hits >= t0.n_hits)
    same_n = t1.n_hits == t0.n_hits
    assert np.all(t1.chi2[same_n] <= t0.chi2[same_n])
    n_cmp = 0
    for e in range(b.n_events):
        lo, hi = int(h.hit_offsets[e * 64]), int(h.hit_offsets[(e + 1) * 64])
        for k in range(int(b.velo_offsets[e]), int(b.velo_offsets[e + 1])):
            ref = brute_force64(h, lo, hi, geom, p1, float(b.velo_x[k]), float(b.velo_y[k]), float(b.velo_tx[k]),
                                float(b.velo_ty[k]))
            if ref is None:
                assert t1.n_hits[k] == 0
                continue
            if np.isfinite(t1.runner_chi2[k]) and abs(t1.runner_chi2[k] - t1.chi2[k]) <= 1e-4 * t1.chi2[k]:
                continue
            assert tuple(t1.hit_idx[:, k]) == ref[0] and t1.n_hits[k] == ref[1]
            n_cmp += 1
    assert n_cmp >= 60


def test_both_directions_changes_few_tracks(wl):
    """On min-bias-like events the mode matters for a fraction of a per cent of the tracks, never lowers n_hits and
    never finds fewer tracklets."""
    import dataclasses
    geom, b, p0 = wl(2, 30)
    _, t0 = run(b, geom, p0, 0)
    _, t1 = run(b, geom, dataclasses.replace(p0, both_directions=1), 0)
    diff = (t1.hit_idx != t0.hit_idx).any(axis=0)
    assert 0 < diff.sum() < 0.01 * diff.size
    assert np.array_equal(t0.n_hits > 0, t1.n_hits > 0) and np.all(t1.n_hits >= t0.n_hits)
