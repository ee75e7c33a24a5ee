"""Test helpers: hand-built hit containers and a float64 brute-force Compass used to pin the oracle."""
import itertools

import numpy as np

import oracle
from synth import geometry as G


def make_hits(geom, per_layer):
    """per_layer[l] = list of (x_at_y0, y_begin, y_end) -> oracle.Hits of ONE event.
    Each hit goes to the column group whose [group_xmin, group_xmax] centre is nearest."""
    rows = []
    for l in range(4):
        for (x, yb, ye) in per_layer[l]:
            g0 = l * 16
            ctr = 0.5 * (geom.group_xmin[g0:g0 + 16].astype(np.float64) + geom.group_xmax[g0:g0 + 16])
            g = g0 + int(np.argmin(np.abs(ctr - x)))
            assert geom.group_xmin[g] <= np.float32(x) <= geom.group_xmax[g]
            rows.append((g, np.float32(x), np.float32(yb), np.float32(ye), l))
    rows.sort(key=lambda r: (r[0], r[1]))
    n = len(rows)
    f = lambda vals: np.asarray(vals, dtype=np.float32).reshape(n)
    offs = np.zeros(65, np.uint32)
    for r in rows:
        offs[r[0] + 1:] += 1
    lay = [r[4] for r in rows]
    return oracle.Hits(
        x_at_y0=f([r[1] for r in rows]), z_at_y0=f([G.LAYER_Z[l] for l in lay]), y_begin=f([r[2] for r in rows]),
        y_end=f([r[3] for r in rows]), dxdy=f([G.LAYER_DXDY[l] for l in lay]),
        weight=f([12.0 / G.PITCH ** 2] * n), id=np.arange(n, dtype=np.uint32), hit_offsets=offs, status=0, n_hits=n)


def run_one(hits, geom, params, velo, mode=0):
    """velo = list of (x, y, tx, ty) at z = 770 for one event."""
    v = np.asarray(velo, dtype=np.float32).reshape(-1, 4)
    vo = np.array([0, len(v)], np.uint32)
    return oracle.compass(hits, v[:, 0].copy(), v[:, 1].copy(), v[:, 2].copy(), v[:, 3].copy(), 770.0, vo, 1,
                          geom, params, mode)


def brute_force64(hits, lo, hi, geom, p, vx, vy, vtx, vty, vz=770.0):
    """float64, lstsq-based exhaustive Compass for ONE track over hits [lo, hi) of its event
    (SURVEY.md 8(c) steps 1-7 with no window search, no cap, no seeding order).
    Returns (hit tuple with -1 = none, n, chi2, qop) or None."""
    x = hits.x_at_y0.astype(np.float64); z = hits.z_at_y0.astype(np.float64)
    yb = hits.y_begin.astype(np.float64); ye = hits.y_end.astype(np.float64)
    sl = hits.dxdy.astype(np.float64); w = hits.weight.astype(np.float64)
    cand = [[] for _ in range(4)]
    for h in range(lo, hi):
        l = int(np.argmin(np.abs(np.asarray(G.LAYER_Z) - z[h])))
        dzv = float(geom.layer_z[l]) - vz
        xe, yex = vx + vtx * dzv, vy + vty * dzv
        d = x[h] + sl[h] * yex - xe
        if abs(d) <= p.win_half[l] and yb[h] - p.y_tol <= yex <= ye[h] + p.y_tol:
            cand[l].append((h, d))
    if sum(1 for c in cand if c) < p.min_hits:
        return None
    res = {}
    for direction, (LA, LB, LC, LD) in enumerate(((0, 2, 1, 3), (3, 1, 2, 0))):
        best = None
        for combo in itertools.product(*[[None] + c for c in cand]):
            n = sum(c is not None for c in combo)
            if n < p.min_hits or combo[LA] is None or combo[LB] is None:
                continue
            (ha, da), (hb, db) = combo[LA], combo[LB]
            bs = (db - da) / (z[hb] - z[ha])
            a0 = da - bs * (z[ha] - p.z_mag)
            if abs(bs) > p.max_slope or abs(a0) > p.kink_tol:
                continue
            ok = True
            for L in (LC, LD):
                if combo[L] is not None:
                    hc, dc = combo[L]
                    ok &= abs(dc - (da + bs * (z[hc] - z[ha]))) <= p.seed_tol
            if not ok:
                continue
            pts = [(0.0, 0.0, p.w_velo)] + [(z[c[0]] - p.z_mag, c[1], w[c[0]]) for c in combo if c is not None]
            dz_, d_, w_ = (np.array(v) for v in zip(*pts))
            A = np.stack([np.ones_like(dz_), dz_], axis=1) * np.sqrt(w_)[:, None]
            sol, *_ = np.linalg.lstsq(A, d_ * np.sqrt(w_), rcond=None)
            chi2 = float((w_ * (d_ - sol[0] - sol[1] * dz_) ** 2).sum())
            if chi2 > p.max_chi2_ndf * (n - 1):
                continue
            key = (-n, chi2, tuple(c[0] if c is not None else 2 ** 31 - 1 for c in combo))
            if best is None or key < best[0]:
                best = (key, tuple(c[0] if c is not None else -1 for c in combo), n, chi2, sol[1] / p.kappa)
        res[direction] = best
    if getattr(p, "both_directions", 0) and res[0] is not None and res[1] is not None:
        best = min(res[0], res[1], key=lambda r: r[0])        # 8(f) row 4: best of both directions, same order
    else:
        best = res[0] if res[0] is not None else res[1]        # A11
    return None if best is None else best[1:]
