"""Hand-built adversarial cases shared by tests/test_oracle_boundaries.py (CPU: the oracle alone must decide as the
construction predicts -- a pin of the oracle's exact-boundary behaviour on raw-bank inputs) and
tests/test_gpu_adversarial.py (GPU == oracle bit for bit on the same inputs, and the same predictions).

Raw banks and VELO states put the path exactly ON the boundaries of the method's predicates (SURVEY.md 8(c) steps
2-7) and one ulp either side, and build exact |d| and chi2 ties.  Inputs are exact by
construction: in an X layer x = x_left + (strip + 0.25 + 0.5 frac) * 0.1875 is a dyadic rational, a VELO state with
tx = ty = 0 extrapolates to (x_v, y_v) unchanged, and the tolerances are inputs (compass_config), so a tolerance can
be set to the very fp32 value a residual takes.  Where a case needs a residual of the method (a seed slope, a kink
intercept) it evaluates that ONE expression in numpy float32 to choose the input; the assertions are on what the
implementation under test then decides.  `run(geom, batch, params)` returns (oracle.Hits, oracle.Tracks)."""
import dataclasses

import numpy as np

import oracle
import synth
from synth import geometry as G
from synth.events import assemble_batch, encode_event

F = np.float32
COL, ROW = 10, 9                       # sector column / row used by the hand-built cases (x_left 192, y 192..288)
X_LEFT = G.X_MIN + G.SECTOR_W * COL


def loose(**kw):
    """Every cut wide open except the ones a test sets: the construction decides what survives."""
    p = synth.make_compass_params(max_candidates_per_layer=16)
    base = dict(win_half=(F(8.0), F(20.0), F(20.0), F(20.0)), y_tol=F(0.5), max_slope=F(10.0), kink_tol=F(1e4),
                seed_tol=F(1e3), max_chi2_ndf=F(1e12))
    base.update(kw)
    return dataclasses.replace(p, **base)


def sector(layer, col=COL, row=ROW):
    return G.dense_sector(layer, col, row)


def x_of(strip, frac=0):
    """x_at_y0 of an X-layer hit, exact in fp32 (and the x of a stereo hit at its sector's y centre)."""
    return F(X_LEFT + (strip + 0.25 + 0.5 * frac) * G.PITCH)


def build(geom, hits, velo):
    """hits: list of (dense sector, strip, frac); velo: list of (x, y, tx, ty) -> one-event synth.Batch."""
    sec = np.array([h[0] for h in hits], np.int64)
    raw, offs = encode_event(geom, sec, np.array([h[1] for h in hits]), np.array([h[2] for h in hits]),
                             np.zeros(len(hits), int), None)
    v = np.asarray(velo, dtype=np.float32).reshape(-1, 4)
    ev = dict(raw=raw, bank_offs=offs, velo=tuple(np.ascontiguousarray(v[:, k]) for k in range(4)),
              truth_hit_id=np.full((len(v), 4), -1, np.int64), q=np.zeros(len(v), np.int8), p=np.zeros(len(v)),
              n_hits=len(hits))
    return assemble_batch(geom, [ev])


def hit_index(geom, h, sec, strip):
    idx = np.nonzero(h.id[:h.n_hits] == ((int(geom.sector_raw_id[sec]) << 9) | strip))[0]
    assert idx.size == 1
    return int(idx[0])


def ulp_steps(v, k):
    v = F(v)
    for _ in range(abs(k)):
        v = np.nextafter(v, F(np.inf) if k > 0 else F(-np.inf))
    return v


def stereo_at(geom, layer, strip, y_e):
    """fp32 value the method gives a stereo hit at y_e: fl(x_at_y0 + fl(dxdy * y_e)), x_at_y0 as the decode
    definition computes it.  Used to choose inputs only."""
    s = sector(layer)
    t = F(F(F(2 * strip) * F(0.5)) + F(0.25))
    x = F(geom.x0[s] + F(t * geom.pitch[s]))
    return F(x + F(geom.dxdy[s] * F(y_e)))


# ---------------------------------------------------------------------------------------------------
# step 2: |d| == win_half[l] exactly and one ulp either side; y_e == y_end + y_tol / y_begin - y_tol
# ---------------------------------------------------------------------------------------------------
def case_window_edge_exact(run, geom, layer):
    y = F(240.0)
    hits = [(sector(l), 100, 0) for l in range(4)]
    D = F(8.0)
    a = x_of(100) if layer in (0, 3) else stereo_at(geom, layer, 100, y)       # fl(x + dxdy*y_e) of the edge hit
    velo, expect = [], []
    for sign in (+1, -1):
        for k in (0, -1, +1, -2, +2):
            vx = ulp_steps(F(a - sign * D), k)
            d = F(a - vx)                                   # exact (Sterbenz): the residual the method computes
            velo.append((vx, y, 0.0, 0.0))
            expect.append(4 if abs(d) <= D else 3)
    assert expect.count(3) >= 4 and expect.count(4) >= 6 and abs(F(a - F(a - D))) == D
    win = [F(20.0)] * 4
    win[layer] = D
    b = build(geom, hits, velo)
    _, t = run(geom, b, loose(win_half=tuple(win)))
    assert t.n_hits.tolist() == expect
    assert np.all((t.hit_idx[layer] >= 0) == (np.array(expect) == 4))


def case_y_edge_exact(run, geom, layer):
    """y_e == y_end + y_tol and y_e == y_begin - y_tol are inside, one ulp further is outside.  The three other
    layers have their hit in the neighbouring row, which contains y_e comfortably."""
    y_tol = F(0.5)
    for edge, other_row in ((F(G.Y_MIN + G.SECTOR_H * (ROW + 1)) + y_tol, ROW + 1),
                            (F(G.Y_MIN + G.SECTOR_H * ROW) - y_tol, ROW - 1)):
        hits = [(sector(l, row=ROW if l == layer else other_row), 200, 1) for l in range(4)]
        velo, expect = [], []
        for k in (0, -1, +1, -3, +3):
            vy = ulp_steps(edge, k)
            inside = (vy <= edge) if other_row == ROW + 1 else (vy >= edge)
            velo.append((x_of(200, 1), vy, 0.0, 0.0))
            expect.append(4 if inside else 3)
        b = build(geom, hits, velo)
        _, t = run(geom, b, loose(win_half=(F(20.0),) * 4, y_tol=y_tol))
        assert t.n_hits.tolist() == expect
        assert np.all((t.hit_idx[layer] >= 0) == (np.array(expect) == 4))


# ---------------------------------------------------------------------------------------------------
# step 5: seed slope, kink intercept and seed_tol exactly at the limit (the limit is an input: it is set to
# the fp32 value the expression takes, then moved by one ulp)
# ---------------------------------------------------------------------------------------------------
def _seed_numbers(geom, strips, vx, y):
    """d per layer and the step-5 expressions of the forward seed (L0, L2), evaluated once in fp32 in the order
    DESIGN.md section 3 writes them."""
    d = [F((x_of(strips[l]) if l in (0, 3) else stereo_at(geom, l, strips[l], y)) - F(vx)) for l in range(4)]
    z = [F(v) for v in G.LAYER_Z]
    zm = F(synth.events.Z_MAG)
    bs = F(F(d[2] - d[0]) / F(z[2] - z[0]))
    a0 = F(d[0] - F(bs * F(z[0] - zm)))
    r1 = abs(F(d[1] - F(d[0] + F(bs * F(z[1] - z[0])))))
    r3 = abs(F(d[3] - F(d[0] + F(bs * F(z[3] - z[0])))))
    return d, bs, a0, r1, r3


def case_seed_cut_edges(run, geom):
    y, vx = F(240.0), F(X_LEFT + 20.0)
    strips = (110, 121, 131, 136)                  # a bent tracklet: residuals of a few mm, all different
    d, bs, a0, r1, r3 = _seed_numbers(geom, strips, vx, y)
    assert bs != 0 and a0 != 0 and r1 > 0 and r3 > 0 and r1 != r3
    three = [(sector(l), strips[l], 0) for l in range(3)]                  # L0, L1, L2 only: forward or nothing
    b3 = build(geom, three, [(vx, y, 0.0, 0.0)])
    four = three + [(sector(3), strips[3], 0)]
    b4 = build(geom, four, [(vx, y, 0.0, 0.0)])
    lo = lambda v: np.nextafter(F(v), F(0.0))
    for p, want in ((loose(max_slope=abs(bs)), 3), (loose(max_slope=lo(abs(bs))), 0),
                    (loose(kink_tol=abs(a0)), 3), (loose(kink_tol=lo(abs(a0))), 0),
                    (loose(seed_tol=r1), 3), (loose(seed_tol=lo(r1)), 0)):
        _, t = run(geom, b3, p)
        assert t.n_hits.tolist() == [want], (p, want)
    # four layers: the L1 / L3 hit drops out of the forward tracklet exactly when its residual passes seed_tol
    big, small = (r1, r3) if r1 > r3 else (r3, r1)
    for p, want in ((loose(seed_tol=big), 4), (loose(seed_tol=lo(big)), 3), (loose(seed_tol=small), 3)):
        _, t = run(geom, b4, p)
        assert t.n_hits.tolist() == [want], (p, want)


def case_chi2_cut_edge(run, geom):
    """chi2 == max_chi2_ndf * (n - 1) is valid, one ulp below the tracklet is dropped (n = 3: the product is exact)."""
    y, vx = F(240.0), F(X_LEFT + 20.0)
    hits = [(sector(0), 110, 0), (sector(1), 117, 1), (sector(2), 131, 0)]
    b = build(geom, hits, [(vx, y, 0.0, 0.0)])
    _, t = run(geom, b, loose())
    chi2 = F(t.chi2[0])
    assert t.n_hits.tolist() == [3] and chi2 > 0
    _, t = run(geom, b, loose(max_chi2_ndf=F(chi2 / F(2.0))))
    assert t.n_hits.tolist() == [3] and t.chi2[0] == chi2
    _, t = run(geom, b, loose(max_chi2_ndf=np.nextafter(F(chi2 / F(2.0)), F(0.0))))
    assert t.n_hits.tolist() == [0]


# ---------------------------------------------------------------------------------------------------
# step 3: exact |d| ties at the candidate cap; step 7: bit-identical chi2 from different seeds / lanes
# ---------------------------------------------------------------------------------------------------
def case_abs_d_ties_at_the_cap(run, geom):
    """Layer 0 holds four hits with |d| = 0.375 exactly (two rows that both contain y_e, strips s-2 and s+2) and
    two farther ones; with C = 2 the cap keeps the two LOWEST hit indices of the tie (both at d = -0.375) although
    the other layers prefer d = +0.375."""
    y = F(G.Y_MIN + G.SECTOR_H * (ROW + 1) + 0.25)                      # inside row ROW (+ y_tol) and row ROW+1
    s0 = 200
    vx = x_of(s0)
    l0 = [(sector(0, row=r), s, 0) for s in (s0 - 2, s0 + 2, s0 + 5, s0 - 6) for r in (ROW, ROW + 1)]
    # the other layers lie on a line through the kick plane that passes d = +0.375 at layer 0
    zm = synth.events.Z_MAG
    others = []
    y_c = G.Y_MIN + G.SECTOR_H * (ROW + 1.5)                             # centre of the row the other hits sit in
    for l in (1, 2, 3):
        want = 0.375 * (G.LAYER_Z[l] - zm) / (G.LAYER_Z[0] - zm)
        stereo = G.LAYER_DXDY[l] * (float(y) - y_c)                       # d = (s - s0) * pitch + dxdy * (y_e - y_c)
        others.append((sector(l, row=ROW + 1), s0 + int(round((want - stereo) / G.PITCH)), 0))
    b = build(geom, l0 + others, [(vx, y, 0.0, 0.0)])
    for C, n_l0 in ((2, 2), (3, 3), (5, 5), (16, 8)):
        p = dataclasses.replace(loose(win_half=(F(8.0), F(30.0), F(30.0), F(30.0))), max_candidates_per_layer=C)
        h, t = run(geom, b, p)
        i = [hit_index(geom, h, sector(0, row=r), s) for s in (s0 - 2, s0 + 2) for r in (ROW, ROW + 1)]
        assert i == sorted(i) and i[1] == i[0] + 1 and i[3] == i[2] + 1
        kept = [v for v in t.cand_list[0, 0].tolist() if v >= 0]
        assert len(kept) == n_l0 and kept == sorted(kept)
        if C == 2:
            assert kept == i[:2] and t.hit_idx[0, 0] == i[0]           # d = -0.375 although +0.375 fits better
        if C == 3:
            assert kept == i[:3] and t.hit_idx[0, 0] == i[2]
        if C >= 5:
            assert t.hit_idx[0, 0] == i[2]                             # lower index of the two d = +0.375 hits
        assert t.n_hits.tolist() == [4]


def case_exact_chi2_ties_across_lanes(run, geom):
    """Twin hits in the two X layers (same strip in two rows that both contain y_e: identical x, z, weight; a
    stereo layer has no exact twins, its x0 differs from row to row): four 4-hit tracklets with bit-identical chi2,
    from different forward seeds (L0 twins), from the combinations of one seed (L3 twins) and, with both
    directions, from different backward seeds.  Step 7 keeps the lowest hit-index tuple; several tracks share the
    batch so that the twins sit in different lanes."""
    y = F(G.Y_MIN + G.SECTOR_H * (ROW + 1) + 0.25)
    strips = (200, 225, 160, 211)
    hits = [(sector(l, row=r), strips[l], 1) for l in (0, 3) for r in (ROW + 1, ROW)]
    hits += [(sector(l, row=ROW + 1), strips[l], 1) for l in (1, 2)]
    velo = [(F(x_of(200) - F(0.1 * k)), y, 0.0, 0.0) for k in range(11)]
    b = build(geom, hits, velo)
    for both in (0, 1):
        h, t = run(geom, b, dataclasses.replace(loose(), both_directions=both))
        low = [hit_index(geom, h, sector(l, row=ROW), strips[l]) for l in (0, 3)]
        high = [hit_index(geom, h, sector(l, row=ROW + 1), strips[l]) for l in (0, 3)]
        assert all(a + 1 == c for a, c in zip(low, high))
        assert np.all(t.n_hits == 4)
        assert np.all(t.hit_idx[0] == low[0]) and np.all(t.hit_idx[3] == low[1])
        assert np.all(t.runner_chi2 == t.chi2)                          # the runner-up really is an exact tie


