"""Pins of the position-dependent kick table in the oracle (A24)."""
import dataclasses

import numpy as np
import pytest

import oracle
import synth
from helpers import brute_force64
from synth.events import EventModel, generate_batch


def lut_geometry(**kw):
    g = synth.make_geometry()
    g.kick = synth.make_kick_lut(**kw)
    return g


def test_constant_table_is_the_constant_kick(wl):
    geom, b, p = wl(2, 15)
    g2 = synth.make_geometry()
    lut = synth.make_kick_lut()
    g2.kick = dataclasses.replace(lut, kappa=np.full_like(lut.kappa, p.kappa), z_mag=np.full_like(lut.z_mag, p.z_mag))
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events)
    t0, t1 = oracle.compass(h, *args, geom, p), oracle.compass(h, *args, g2, p)
    assert np.array_equal(t0.hit_idx, t1.hit_idx) and np.array_equal(t0.qop.view(np.uint32), t1.qop.view(np.uint32))
    assert np.array_equal(t0.chi2.view(np.uint32), t1.chi2.view(np.uint32))


def test_cell_lookup(wl):
    """kappa[cell] = 100 + cell and a constant kick plane: q/p = b / kappa gives the cell every track looked up.
    Interior positions against a float64 bin index, positions outside the table clamp, NaN takes cell 0."""
    geom, b, p = wl(2, 20)
    lut = synth.make_kick_lut(half_x=250.0, half_y=200.0)            # smaller than the acceptance: some look-ups clamp
    code = (100.0 + np.arange(lut.nx * lut.ny)).astype(np.float32)
    g2 = synth.make_geometry()
    g2.kick = dataclasses.replace(lut, kappa=code, z_mag=np.full_like(lut.z_mag, p.z_mag))
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, geom, b.hit_capacity)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events)
    t0, t1 = oracle.compass(h, *args, geom, p), oracle.compass(h, *args, g2, p)
    assert np.array_equal(t0.hit_idx, t1.hit_idx) and np.array_equal(t0.chi2.view(np.uint32), t1.chi2.view(np.uint32))
    ok = (t0.n_hits > 0) & (np.abs(t0.qop) > 1e-7)
    cell = np.rint(p.kappa * t0.qop[ok].astype(np.float64) / t1.qop[ok].astype(np.float64) - 100.0).astype(int)
    dzr = lut.z_ref - b.velo_z
    xk = b.velo_x[ok].astype(np.float64) + b.velo_tx[ok].astype(np.float64) * dzr
    yk = b.velo_y[ok].astype(np.float64) + b.velo_ty[ok].astype(np.float64) * dzr
    u, v = (xk - lut.x_lo) * lut.inv_dx, (yk - lut.y_lo) * lut.inv_dy
    interior = (np.abs(u - np.rint(u)) > 1e-3) & (np.abs(v - np.rint(v)) > 1e-3)        # away from bin edges
    want = lut.cell64(xk, yk)
    assert interior.sum() > 1500 and np.array_equal(cell[interior], want[interior])
    assert len(np.unique(cell)) > 40                                  # many different cells were hit
    outside = (np.abs(xk) > 250.0) | (np.abs(yk) > 200.0)
    assert outside.sum() > 20                                         # clamped look-ups are in the sample


def test_per_track_kick_against_float64_search(wl):
    """An independent float64 exhaustive search (numpy lstsq) run with each track's own (kappa, z_mag) picks the
    tracklets the oracle picks with the table."""
    g = lut_geometry(bow=120.0, falloff=0.3)                          # a strongly varying table
    b = generate_batch(g, EventModel(fixed_tracks=25, efficiency=1.0, noise_mean=30.0), seed=11, n_events=2)
    p = synth.make_compass_params()
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, g, b.hit_capacity)
    t = oracle.compass(h, b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events, g, p)
    lut = g.kick
    n_checked = 0
    for e in range(2):
        lo, hi = int(h.hit_offsets[64 * e]), int(h.hit_offsets[64 * (e + 1)])
        for k in range(int(b.velo_offsets[e]), int(b.velo_offsets[e + 1])):
            dzr = lut.z_ref - b.velo_z
            cell = int(lut.cell64(b.velo_x[k] + b.velo_tx[k] * dzr, b.velo_y[k] + b.velo_ty[k] * dzr))
            pk = dataclasses.replace(p, kappa=float(lut.kappa[cell]), z_mag=float(lut.z_mag[cell]))
            want = brute_force64(h, lo, hi, g, pk, float(b.velo_x[k]), float(b.velo_y[k]), float(b.velo_tx[k]), float(b.velo_ty[k]))
            if want is None:
                assert t.n_hits[k] == 0
                continue
            assert tuple(t.hit_idx[:, k]) == want[0] and t.n_hits[k] == want[1]
            assert abs(t.chi2[k] - want[2]) <= 2e-3 * max(want[2], 1e-3) + 1e-4
            assert abs(t.qop[k] - want[3]) <= 1e-4 * abs(want[3]) + 1e-9
            n_checked += 1
    assert n_checked >= 30


def test_momentum_is_unbiased_only_with_the_table():
    """Tracks bent by the table: q/p from the table's kappa is unbiased and has the charge right; the constant
    60 MeV overestimates |q/p| where the integrated field is weaker."""
    g = lut_geometry(falloff=0.3, half_x=300.0, half_y=250.0)
    b = generate_batch(g, EventModel(mean_tracks=150.0, efficiency=1.0, noise_mean=200.0), seed=12, n_events=30)
    p = synth.make_compass_params()
    h = oracle.decode(b.raw, b.bank_offsets, b.n_events, g, b.hit_capacity)
    args = (b.velo_x, b.velo_y, b.velo_tx, b.velo_ty, b.velo_z, b.velo_offsets, b.n_events)
    with_lut = oracle.compass(h, *args, g, p)
    const = oracle.compass(h, *args, synth.make_geometry(), p)
    m = synth.physics_metrics(b.truth_hit_id, b.truth_q, h.id[:h.n_hits], with_lut.hit_idx, with_lut.n_hits, with_lut.qop)
    assert m["efficiency"] > 0.97 and m["charge_ok"] == 1.0
    lut = g.kick
    dzr = lut.z_ref - b.velo_z
    kap = lut.kappa[lut.cell64(b.velo_x + b.velo_tx * dzr, b.velo_y + b.velo_ty * dzr)]
    sel = (with_lut.n_hits == 4) & (const.n_hits == 4) & (b.truth_p > 3e3) & (b.truth_p < 2e4) & (kap < 54.0)
    assert sel.sum() > 150
    r_lut = with_lut.qop[sel] * b.truth_p[sel] * b.truth_q[sel] - 1.0
    r_const = const.qop[sel] * b.truth_p[sel] * b.truth_q[sel] - 1.0
    assert abs(np.median(r_lut)) < 0.01
    assert np.median(r_const) < -0.05                                  # kappa too large -> |q/p| too small
