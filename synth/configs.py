"""The five workloads of BASELINE.json ``configs`` and the Compass parameter sets.

``CompassParams`` is INPUT data for both implementations: every derived field
(``win_half``, ``max_slope``) is computed here once, in float64, and rounded to
float32 once, so neither side re-derives it.
The paper prints no tolerance values (its knobs are "number of sectors" and
"number of candidates"); the defaults are SURVEY.md A8's.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

from . import geometry as G
from .events import EventModel, Batch, generate_batch, KAPPA, Z_MAG


@dataclass(frozen=True)
class CompassParams:
    win_half: tuple            # 4 x f32, half-width of the x window per layer [mm]
    y_tol: float
    max_slope: float           # |seed slope - VELO slope| limit
    kink_tol: float            # |intercept of the seed line at z_mag| limit [mm]
    seed_tol: float            # |residual to the seed line| limit in the other two layers [mm]
    w_velo: float              # weight of the VELO pseudo-point [mm^-2]
    max_chi2_ndf: float
    kappa: float               # MeV
    z_mag: float               # mm
    min_hits: int              # 3 or 4
    max_candidates_per_layer: int
    both_directions: int = 0   # 0: backward seeds only if forward found nothing (A11); 1: best of both directions


def make_compass_params(p_min_gev: float = 2.0, window_scale: float = 1.0, min_hits: int = 3,
                        max_candidates_per_layer: int = 16, x_tol0: float = 0.5, y_tol: float = 0.5,
                        slope_tol: float = 0.0015, kink_tol: float = 1.5, seed_tol: float = 0.5,
                        w_velo: float = 100.0, max_chi2_ndf: float = 9.0, both_directions: int = 0) -> CompassParams:
    f = lambda v: float(np.float32(v))
    kick = window_scale * KAPPA / (p_min_gev * 1e3)          # max |slope change| at p_min, scaled
    win = tuple(f(kick * (z - Z_MAG) + x_tol0) for z in G.LAYER_Z)
    return CompassParams(
        win_half=win, y_tol=f(y_tol), max_slope=f(kick + slope_tol), kink_tol=f(kink_tol),
        seed_tol=f(seed_tol), w_velo=f(w_velo), max_chi2_ndf=f(max_chi2_ndf), kappa=f(KAPPA),
        z_mag=f(Z_MAG), min_hits=int(min_hits), max_candidates_per_layer=int(max_candidates_per_layer),
        both_directions=int(both_directions))


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    n_events: int
    seed: int
    model: EventModel
    p_min_gev: float = 2.0
    window_scale: float = 1.0
    min_hits: int = 3
    max_candidates_per_layer: int = 16

    def compass_params(self, **over) -> CompassParams:
        kw = dict(p_min_gev=self.p_min_gev, window_scale=self.window_scale, min_hits=self.min_hits,
                  max_candidates_per_layer=self.max_candidates_per_layer)
        kw.update(over)
        return make_compass_params(**kw)


_MINBIAS = EventModel(mean_tracks=150.0, efficiency=0.97, noise_mean=1500.0)

CONFIGS = {
    # BASELINE.json configs[0]: tiny single event, noise-free, 20 tracks, seed 1
    1: WorkloadConfig("config1_tiny", 1, 1, EventModel(fixed_tracks=20, efficiency=1.0, noise_mean=0.0)),
    # configs[1]: 100 min-bias-like events, ~2000 hits each, seed 2
    2: WorkloadConfig("config2_minbias100", 100, 2, _MINBIAS),
    # configs[2]: 1000-event throughput batch, seed 3  (the metric's workload)
    3: WorkloadConfig("config3_throughput1000", 1000, 3, _MINBIAS),
    # configs[3]: high occupancy, Poisson(600) tracks, ~8000 hits, p >= 1.5 GeV, C = 32, seed 4
    4: WorkloadConfig("config4_highocc1000", 1000, 4,
                      EventModel(mean_tracks=600.0, efficiency=0.97, noise_mean=6000.0, p_min_gev=2.0),
                      p_min_gev=1.5, max_candidates_per_layer=32),
    # configs[4]: 10000 events for the {min_hits} x {scale} x {C} sweep, seed 5
    5: WorkloadConfig("config5_sweep10000", 10000, 5, _MINBIAS),
}

SWEEP_MIN_HITS = (3, 4)
SWEEP_SCALE = (0.5, 1.0, 2.0)
SWEEP_CANDIDATES = (8, 16, 32)


def make_workload(config: int | WorkloadConfig, n_events: int | None = None, workers: int = 1,
                  first_event: int = 0):
    """(geometry, batch, params) for one of the five configs (optionally fewer events)."""
    cfg = CONFIGS[config] if isinstance(config, int) else config
    geom = G.make_geometry()
    n = cfg.n_events if n_events is None else n_events
    batch = generate_batch(geom, cfg.model, cfg.seed, n, first_event=first_event, workers=workers)
    return geom, batch, cfg.compass_params()
