"""Scoring against generator truth.

reconstructible = truth track with recorded hits in >= 3 of the 4 layers;
a tracklet is matched if >= 70 % of its hits belong to its VELO track's particle;
efficiency = matched & reconstructible / reconstructible; ghost (fake) rate = unmatched / all
tracklets; clone rate is 0 by construction (one tracklet per VELO track).
"""
from __future__ import annotations

import numpy as np


def physics_metrics(truth_hit_id: np.ndarray, truth_q: np.ndarray, hit_id: np.ndarray,
                    trk_hit_idx: np.ndarray, trk_n_hits: np.ndarray, trk_qop: np.ndarray) -> dict:
    """truth_hit_id [T,4] (i64, -1 none); hit_id [H] decoded ids; trk_hit_idx [4,T] global hit index or -1."""
    T = truth_hit_id.shape[0]
    idx = np.asarray(trk_hit_idx).reshape(4, T).T.astype(np.int64)      # [T,4]
    has = idx >= 0
    ids = np.where(has, np.asarray(hit_id, dtype=np.int64)[np.clip(idx, 0, max(len(hit_id) - 1, 0))], -2) \
        if len(hit_id) else np.full((T, 4), -2, dtype=np.int64)
    n = np.asarray(trk_n_hits).astype(np.int64)
    good = (ids == truth_hit_id) & has
    n_good = good.sum(axis=1)
    found = n > 0
    matched = found & (n_good * 10 >= 7 * np.maximum(n, 1))
    reconstructible = (truth_hit_id >= 0).sum(axis=1) >= 3
    n_rec = int(reconstructible.sum())
    n_found = int(found.sum())
    sign_ok = np.sign(np.asarray(trk_qop)) == np.asarray(truth_q)
    return dict(
        n_tracks=int(T), n_reconstructible=n_rec, n_tracklets=n_found,
        n_matched=int(matched.sum()),
        efficiency=float((matched & reconstructible).sum() / n_rec) if n_rec else float("nan"),
        ghost_rate=float((found & ~matched).sum() / n_found) if n_found else float("nan"),
        charge_ok=float((sign_ok & matched).sum() / max(int(matched.sum()), 1)),
        four_hit_fraction=float((n == 4).sum() / n_found) if n_found else float("nan"),
    )
