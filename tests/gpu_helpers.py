"""Runs a synth.Batch through the C ABI (binding -> libutcompass.so) and returns numpy views."""
import numpy as np


class GpuRunner:
    def __init__(self, geom_tables):
        import torch
        from paper_2002_11529_b200 import binding as B
        self.B, self.torch = B, torch
        self.geom = B.ut_geometry_upload(geom_tables)
        self.tables = geom_tables

    def decode(self, raw, bank_offsets, n_events, capacity):
        B, torch = self.B, self.torch
        hits = B.Hits(capacity, max(n_events, 1), self.geom)
        raw_d = B.to_device_raw(raw)
        bo_d = B.to_device_u32(bank_offsets)
        B.ut_decode(raw_d, bo_d, n_events, self.geom, hits)
        torch.cuda.synchronize()
        self._keep = (raw_d, bo_d)
        return hits

    def hits_numpy(self, hits, n_events):
        off = hits.hit_offsets[:n_events * self.geom.n_groups + 1].cpu().numpy().view(np.uint32)
        n = int(off[-1])
        out = {f: getattr(hits, f)[:n].cpu().numpy() for f in hits.FIELDS}
        out["id"] = out["id"].view(np.uint32)
        return out, off, int(hits.status.item()) & 0xFFFFFFFF

    def compass(self, hits, batch, params, n_events=None):
        B, torch = self.B, self.torch
        n_events = batch.n_events if n_events is None else n_events
        velo = B.VeloStates(batch.velo_x, batch.velo_y, batch.velo_tx, batch.velo_ty, batch.velo_z)
        vo = B.to_device_u32(batch.velo_offsets)
        tracks = B.Tracks(int(batch.velo_offsets[n_events]))
        B.compass_track(hits, hits.hit_offsets, velo, vo, n_events, B.make_config(params), tracks)
        torch.cuda.synchronize()
        idx, n, qop, chi2 = tracks.numpy()
        return dict(hit_idx=idx, n_hits=n, qop=qop, chi2=chi2, status=int(tracks.status.item()) & 0xFFFFFFFF)

    def run(self, batch, params):
        hits = self.decode(batch.raw, batch.bank_offsets, batch.n_events, batch.hit_capacity)
        trk = self.compass(hits, batch, params)
        return hits, trk


def compare_decode(ref, got, off_got, status_got):
    """ref: oracle.Hits; got: dict of numpy arrays.  Bit-exact (north_star)."""
    assert status_got == ref.status
    assert np.array_equal(off_got, ref.hit_offsets)
    n = ref.n_hits
    for f in ("x_at_y0", "z_at_y0", "y_begin", "y_end", "dxdy", "weight"):
        a, b = getattr(ref, f)[:n].view(np.uint32), got[f][:n].view(np.uint32)
        assert np.array_equal(a, b), f"{f}: {np.nonzero(a != b)[0][:10]}"
    assert np.array_equal(ref.id[:n], got["id"][:n])


def compare_tracks(ref, got, rel=1e-5, status=0):
    """ref: oracle.Tracks.  Hit indices exact except flagged near-ties (<= 1e-5 relative between the two
    best chi2 of the same n); q/p and chi2 within 1e-5 relative.  Returns the number of flagged tracks."""
    assert got["status"] == status
    near_tie = np.isfinite(ref.runner_chi2) & (np.abs(ref.runner_chi2 - ref.chi2) <= rel * np.abs(ref.chi2))
    same_idx = np.all(ref.hit_idx == got["hit_idx"], axis=0)
    bad = ~same_idx & ~near_tie
    assert not bad.any(), f"hit index mismatch on tracks {np.nonzero(bad)[0][:10]}"
    assert np.array_equal(ref.n_hits[~near_tie], got["n_hits"][~near_tie])
    ok = same_idx
    assert np.allclose(got["qop"][ok], ref.qop[ok], rtol=rel, atol=0)
    assert np.allclose(got["chi2"][ok], ref.chi2[ok], rtol=rel, atol=0)
    return int((~same_idx).sum()), int(near_tie.sum())
