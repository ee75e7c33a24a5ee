"""Hand-built malformed raw batches for the bank rule DESIGN.md A22 (a bank must start on a 4-byte boundary,
hold at least its 6-byte header and lie inside its event's byte range).  Input construction only: the expected
hits are computed from the ENCODER's inputs (which banks survive), never by decoding."""
import numpy as np

from synth.events import encode_event


def _ids(geom, sector, strip):
    return ((geom.sector_raw_id[np.asarray(sector)].astype(np.int64) << 9) | np.asarray(strip)).tolist()


def _random_event(geom, rng, n):
    key = rng.choice(geom.n_sectors * 512, n, replace=False)
    sector, strip = key // 512, key % 512
    frac = rng.integers(0, 2, n)
    order = rng.permutation(geom.n_sectors)
    raw, offs = encode_event(geom, sector, strip, frac, np.zeros(n, int), order)
    return sector, strip, order, raw, offs


def misaligned_tail(geom, seed=11, n=3000):
    """One event.  The 2 pad bytes of the bank at position j (even count) are cut out: bank j is 2 bytes short of
    round4(6 + 2*count) and every later bank starts 2 bytes off a 4-byte boundary while its size is still right.
    Valid banks: positions < j only.  Returns (raw, offs, expected sorted ids, j)."""
    rng = np.random.default_rng(seed)
    sector, strip, order, raw, offs = _random_event(geom, rng, n)
    counts = np.bincount(sector, minlength=geom.n_sectors)[order]           # per bank position
    even = np.nonzero((counts % 2 == 0) & (np.arange(geom.n_sectors) > 300) & (np.arange(geom.n_sectors) < 600))[0]
    j = int(even[0])
    cut = int(offs[j + 1]) - 2
    assert not raw[cut:cut + 2].any()                                        # the pad
    raw2 = np.concatenate([raw[:cut], raw[cut + 2:]])
    offs2 = offs.copy()
    offs2[j + 1:] -= 2
    pos = np.empty(geom.n_sectors, np.int64)
    pos[order] = np.arange(geom.n_sectors)
    keep = pos[sector] < j
    assert keep.sum() > 500 and (~keep).sum() > 500
    return raw2, offs2.astype(np.uint32), sorted(_ids(geom, sector[keep], strip[keep])), j


def foreign_bank(geom, seed=12, n=2500):
    """Two events.  In event 1 the offsets of bank position j and j+1 are redirected to a well-formed bank of the
    SAME sector inside event 0's byte range (aligned, size right, different words).  Positions j-1, j and j+1 of
    event 1 are lost; without the range rule the foreign words would be decoded into event 1.
    Returns (raw, offs, [expected sorted ids event 0, event 1])."""
    rng = np.random.default_rng(seed)
    ns = geom.n_sectors
    s0, t0, o0, raw0, offs0 = _random_event(geom, rng, n)
    s1, t1, o1, raw1, offs1 = _random_event(geom, rng, n)
    pos1 = np.empty(ns, np.int64)
    pos1[o1] = np.arange(ns)
    pos0 = np.empty(ns, np.int64)
    pos0[o0] = np.arange(ns)
    c0 = np.bincount(s0, minlength=ns)
    for j in range(400, 600):
        S = int(o1[j])                                                       # sector of event 1's bank at position j
        if c0[S] >= 2:
            break
    p = int(offs0[pos0[S]])
    size = int(offs0[pos0[S] + 1]) - p
    raw = np.concatenate([raw0, raw1])
    offs = np.concatenate([offs0[:-1], offs1 + raw0.size]).astype(np.int64)
    offs[ns + j] = p
    offs[ns + j + 1] = p + size
    lost = (pos1[s1] >= j - 1) & (pos1[s1] <= j + 1)
    assert lost.sum() >= 1
    return raw, offs.astype(np.uint32), [sorted(_ids(geom, s0, t0)), sorted(_ids(geom, s1[~lost], t1[~lost]))]
